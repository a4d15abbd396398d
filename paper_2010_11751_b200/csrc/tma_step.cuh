// tma_step.cuh -- the stream-and-collide step with its loads staged through shared memory by the
// TMA unit (1-D bulk copies, cp.async.bulk + mbarrier), SoA layout.
//
// Why: in step_kernel (kernels.cuh) every byte in flight occupies a destination register of some
// thread, and the register file caps the bytes in flight below what hides the DRAM latency at full
// bandwidth -- worst in fp32, where a register holds 4 bytes.  Here a block walks a
// sequence of tiles of B consecutive cells; one thread asks the TMA unit for the Q population rows
// (and the code bytes) of the tile S-1 tiles ahead, which land in shared memory without passing
// through registers, and completion is signalled on an mbarrier per stage.  The bytes in flight are
// then (S-1) stages x resident blocks, independent of the register file.
//
// For direction k the tile of cells [base, base+B) needs the contiguous run of B elements that starts
// at element base + ldo[k] of the source array (ldo = the per-direction offset make_args precomputes:
// plane and neighbour shift): a neighbour in y or x shifts the run by whole rows /
// layers, a neighbour in z by one element.  A bulk copy needs 16-byte alignment, so the aligned
// superset of B elements + 16 bytes is copied and thread t reads element (shift_k + t) of the row.
//
// Cells next to a wall or on the periodic seam (link mask, kernels.cuh) do not get their values from
// the runs: a warp that holds such a cell takes the masked path of load_cell straight from global
// memory, exactly as in step_kernel.  Tiles within one neighbour reach of either end of the array
// are not staged at all (their runs would leave the allocation) and take that path too.
// Stores are the per-thread coalesced stores of step_kernel (a store holds no register while in flight).
#pragma once
#include "kernels.cuh"

namespace lbm {

__device__ __forceinline__ unsigned smem_addr(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned bar, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned bar, unsigned parity)
{
    unsigned ok;
    do {
        asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2; selp.u32 %0, 1, 0, p; }"
                     : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    } while (!ok);
}
// global -> shared, `bytes` a multiple of 16, both addresses 16-byte aligned; completes on `bar`
__device__ __forceinline__ void bulk_load(unsigned dst, const void* src, unsigned bytes, unsigned bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
// shared -> global
__device__ __forceinline__ void bulk_store(void* dst, unsigned src, unsigned bytes)
{
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dst), "r"(src), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void bulk_wait_read() { asm volatile("cp.async.bulk.wait_group.read %0;" ::"n"(N) : "memory"); }
__device__ __forceinline__ void fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// geometry of one stage in shared memory
template <class T, int Q, int B>
struct TmaStage {
    static constexpr int E16 = 16 / (int)sizeof(T);              // elements per 16 bytes
    static constexpr int ROW_BYTES = B * (int)sizeof(T) + 16;    // aligned superset of a run of B elements
    static constexpr int CODE_OFF = Q * ROW_BYTES;
    static constexpr int BYTES = (CODE_OFF + B + 127) / 128 * 128;
    static constexpr unsigned TX = Q * ROW_BYTES + B;            // bytes that complete a stage
};

template <class T, int Q, int B, int S>
__host__ __device__ constexpr size_t tma_smem_bytes() { return (size_t)S * TmaStage<T, Q, B>::BYTES + 8 * S + 128; }

// blocks per SM the launch asks for (register cap) and the tile size, per precision and lattice
template <class T, int Q>
__host__ __device__ constexpr int tma_tile() { return sizeof(T) == 4 ? 256 : 128; }
template <class T, int Q>
__host__ __device__ constexpr int tma_stages() { return 3; }
template <class T, int Q>
__host__ __device__ constexpr int tma_min_blocks() { return sizeof(T) == 4 ? (Q == 19 ? 3 : 2) : (Q == 19 ? 3 : 2); }

template <class T, int Q, int MODEL, int LOAD, int STORE>
__global__ void __launch_bounds__((tma_tile<T, Q>()), (tma_min_blocks<T, Q>())) step_kernel_tma(const StepArgs<T> a)
{
    constexpr bool SHIFT = sizeof(T) == 4;
    constexpr int B = tma_tile<T, Q>(), S = tma_stages<T, Q>();
    using St = TmaStage<T, Q, B>;
    extern __shared__ __align__(128) unsigned char smem[];
    const unsigned stage0 = smem_addr(smem);
    const unsigned bar0 = stage0 + S * St::BYTES;   // S mbarriers of 8 bytes

    asm volatile("griddepcontrol.launch_dependents;");   // see step_kernel
    if (threadIdx.x == 0) {
        for (int s = 0; s < S; ++s) mbar_init(bar0 + 8 * s, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    const int n = a.g.n;
    const int ntiles = (n + B - 1) / B;
    // a tile is staged when all its runs lie inside the array: one neighbour reach from both ends
    const long long margin = (long long)a.g.ny * a.g.nz + a.g.nz + 1 + St::E16;
    auto staged = [&](int tile) {
        const long long base = (long long)tile * B;
        return base >= margin && base + B + margin <= (long long)n;
    };
    auto issue = [&](int tile, int s) {   // thread 0 only
        if (!staged(tile)) return;
        const long long base = (long long)tile * B;
        const unsigned bar = bar0 + 8 * s, dst = stage0 + s * St::BYTES;
        mbar_expect_tx(bar, St::TX);
        static_for<Q>([&](auto kc) {
            const long long st = base + a.ldo[kc] / (long long)sizeof(T);     // first element of the run
            const long long lo = st & ~(long long)(St::E16 - 1);
            bulk_load(dst + kc * St::ROW_BYTES, a.src + lo, St::ROW_BYTES, bar);
        });
        bulk_load(dst + St::CODE_OFF, a.code + base, B, bar);
    };

    asm volatile("griddepcontrol.wait;" ::: "memory");   // populations of the previous step are complete
    const int first = blockIdx.x, stride = gridDim.x;
    if (threadIdx.x == 0)
        for (int j = 0; j < S - 1; ++j)
            if (first + j * stride < ntiles) issue(first + j * stride, j);

    unsigned phase = 0;   // bit s = parity of the next completion of stage s (only staged tiles arm a stage)
    int j = 0;
    for (int tile = first; tile < ntiles; tile += stride, ++j) {
        const int s = j % S;
        if (threadIdx.x == 0) {   // refill the stage that was read in the previous iteration (the barrier below has passed)
            const int ahead = tile + (S - 1) * stride;
            if (ahead < ntiles) issue(ahead, (j + S - 1) % S);
        }
        const long long i = (long long)tile * B + threadIdx.x;
        const bool st = staged(tile);
        T f[Q];
        CellState cs;
        if (st) {
            const unsigned char* stage = smem + s * St::BYTES;
            mbar_wait(bar0 + 8 * s, (phase >> s) & 1u);
            phase ^= 1u << s;
            const uint8_t c = stage[St::CODE_OFF + threadIdx.x];
            cs.active = !(c & 3);
            const bool edge = c == CODE_EDGE;
            cs.masked = __any_sync(0xffffffffu, edge);
            cs.partial = __any_sync(0xffffffffu, cs.active) && !cs.active;
            cs.mask = edge ? edge_mask(a.grp, a.mask, i) : 0ull;
            if (cs.active && !cs.masked) {
                const long long base = (long long)tile * B;
                static_for<Q>([&](auto kc) {
                    const long long e0 = base + a.ldo[kc] / (long long)sizeof(T);
                    const int sh = (int)(e0 & (St::E16 - 1));
                    f[kc] = reinterpret_cast<const T*>(stage + kc * St::ROW_BYTES)[sh + threadIdx.x];
                });
            }
        } else {
            cs = cell_state(a, i, n);
        }
        __syncthreads();   // every thread has taken what it needs from the stage
        if (cs.active) {
            if (!st || cs.masked) load_cell<T, Q, true, LOAD>(a, (int)i, cs.masked, cs.mask, f);
            collide<Q, MODEL, SHIFT>(f, a.rt);
            store_cell<T, Q, true, STORE>(a, (int)i, cs.masked, cs.mask, f);
        } else if constexpr (STORE == ST_LOCAL && LOAD != LD_LOCAL) {
            if (cs.partial) {   // two-population: fill the wall lanes' slots of a written sector (see step_kernel)
                char* __restrict__ p = reinterpret_cast<char*>(a.dst + i);
                static_for<Q>([&](auto kc) { *reinterpret_cast<T*>(p + a.sto[kc]) = T(0); });
            }
        }
    }
}

}  // namespace lbm
