// aos_march.cuh -- two-population pull step in the AoS layout with the neighbour records staged in
// shared memory by TMA bulk copies: a block owns a TY x TZ cross-section in (y, z) and MARCHES along x.
//
// Why: in AoS the 19 / 27 values a cell pulls lie in 19 / 27 different records, and a
// warp request for "slot k of 32 consecutive cells" uses 8 of every 32 bytes it moves through L1 / L2;
// ncu shows the gather bound by those sectors, not by DRAM (profiles/r02_aos_*).  A shared-memory tile
// helps only if the neighbour records of a cell are neighbours in the tile.  The x-layers x-1, x, x+1 of
// the (TY+2) x (TZ+2) cross-section around the block's cells are therefore kept resident in a ring of
// four layer buffers: while layer x is computed, the rows of layer x+2 arrive (one cp.async.bulk per row:
// a row segment of records is contiguous in AoS; completion on one mbarrier per buffer).  Every record is
// fetched from L2 once per block that needs it ((TY+2)(TZ+2) / (TY TZ) = 1.6 x the algorithmic reads for
// 4 x 32, fully coalesced) instead of once per value.  Results are collected in a second tile and
// written out as whole rows, coalesced (two-population: the other array, nothing in place).
//
// Only bulk cells take their values from the tile.  Cells with a link mask (next to a wall, on the
// periodic seam) use the masked path of load_cell on global memory, as everywhere else; solid cells of
// the written array get zeros.  The kernel needs the two outermost x-layers to hold no bulk cell's
// neighbour, i.e. no fluid or ghost cell (a cavity, a channel closed in x): the host dispatches it only
// then, and only for the whole lattice.
#pragma once
#include "kernels.cuh"
#include "tma_step.cuh"

namespace lbm {

template <class T, int Q, int TY, int TZ>
struct MarchGeo {
    static constexpr int AL = 16 / (int)sizeof(T);                 // records per aligned unit: AL * Q * sizeof(T) is a multiple of 16
    static constexpr int RW = (TZ + 2 + AL + AL - 1) / AL * AL;    // records per staged row: z0-1 .. z0+TZ plus the alignment shift
    static constexpr int ROW_BYTES = RW * Q * (int)sizeof(T);
    static constexpr int ROWS = TY + 2;
    static constexpr int LAYER_BYTES = (ROWS * ROW_BYTES + 127) / 128 * 128;
    static constexpr int RING = 4;
    static constexpr int OUT_BYTES = (TY * TZ * Q * (int)sizeof(T) + 127) / 128 * 128;
    static constexpr int SMEM = RING * LAYER_BYTES + OUT_BYTES + 64;
};

template <class T, int Q, int MODEL, int TY, int TZ>
__global__ void __launch_bounds__(TY * TZ, 1) step_kernel_aos_march(const StepArgs<T> a, int xlen)
{
    static_assert(TZ == 32, "one warp = one z-row of the tile");
    constexpr bool SHIFT = sizeof(T) == 4;
    using L = Lat<Q>;
    using G = MarchGeo<T, Q, TY, TZ>;
    extern __shared__ __align__(128) unsigned char smem[];
    const unsigned ring0 = smem_addr(smem);
    T* out = reinterpret_cast<T*>(smem + G::RING * G::LAYER_BYTES);
    const unsigned bar0 = ring0 + G::RING * G::LAYER_BYTES + G::OUT_BYTES;

    const int nx = a.g.nx, ny = a.g.ny, nz = a.g.nz;
    const int z0 = blockIdx.x * TZ, y0 = blockIdx.y * TY;
    // this block computes the layers [xs, xe) of 1 .. nx-2
    const int xs = 1 + blockIdx.z * xlen, xe = min(nx - 1, xs + xlen);
    const int lz = threadIdx.x & (TZ - 1), ly = threadIdx.x / TZ;
    const int y = y0 + ly, z = z0 + lz;
    const bool inside = y < ny && z < nz;

    if (threadIdx.x == 0) {
        for (int s = 0; s < G::RING; ++s) mbar_init(bar0 + 8 * s, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    // first record of the staged row j (global row y0-1+j) of layer l, and its aligned start
    auto row_first = [&](int l, int j) -> long long { return ((long long)l * ny + (y0 - 1 + j)) * nz + (z0 - 1); };
    const long long nrec = a.g.n;
    // rows of layer l into ring buffer l % RING; rows that would leave the array are skipped (their
    // records can only be neighbours of face cells, which do not read the tile)
    auto issue = [&](int l) {   // warp 0, lanes 0 .. ROWS-1 issue one row each; lane 0 arms the barrier
        const int s = l & (G::RING - 1);
        const unsigned bar = bar0 + 8 * s;
        const int j = threadIdx.x;
        bool ok = false;
        long long ga = 0;
        if (j < G::ROWS) {
            const int gy = y0 - 1 + j;
            ga = row_first(l, j) & ~(long long)(G::AL - 1);
            ok = gy >= 0 && gy < ny && ga >= 0 && ga + G::RW <= nrec;
        }
        const unsigned rows = __popc(__ballot_sync(0xffffffffu, ok));
        if (j == 0) mbar_expect_tx(bar, rows * (unsigned)G::ROW_BYTES);
        __syncwarp();
        if (ok) bulk_load(ring0 + s * G::LAYER_BYTES + j * G::ROW_BYTES, a.src + ga * Q, G::ROW_BYTES, bar);
    };

    if (threadIdx.x < 32) {
        issue(xs - 1);
        issue(xs);
        if (xs + 1 < nx) issue(xs + 1);
    }
    unsigned phase = 0;
    auto wait_layer = [&](int l) {
        const int s = l & (G::RING - 1);
        mbar_wait(bar0 + 8 * s, (phase >> s) & 1u);
        phase ^= 1u << s;
    };
    wait_layer(xs - 1);
    wait_layer(xs);

    for (int x = xs; x < xe; ++x) {
        if (threadIdx.x < 32 && x + 2 < nx && x + 2 <= xe) issue(x + 2);   // into the buffer of layer x-2, free since the barrier below
        if (x + 1 < nx) wait_layer(x + 1);
        const long long i = ((long long)x * ny + y) * nz + z;
        CellState cs;
        cs.active = false; cs.masked = false; cs.partial = false; cs.mask = 0ull;
        uint8_t c = CODE_WALL;
        if (inside) c = a.code[i];
        cs.active = !(c & 3);
        const bool edge = c == CODE_EDGE;
        if (edge) cs.mask = edge_mask(a.grp, a.mask, i);
        T f[Q];
        T* rec = out + (size_t)threadIdx.x * Q;
        if (cs.active && !edge) {
            static_for<9>([&](auto gc) {
                constexpr int gx = gc / 3 - 1, gy = gc % 3 - 1;
                // f_k(x) = pop_k(x - c_k): the record at (x - gx, y - gy, z - cz), slot of k
                const int l = x - gx, j = ly + 1 - gy;
                const long long g0 = row_first(l, j);
                const int sh = (int)(g0 & (G::AL - 1));
                const T* row = reinterpret_cast<const T*>(smem + (l & (G::RING - 1)) * G::LAYER_BYTES + j * G::ROW_BYTES);
                static_for<3>([&](auto dc) {
                    constexpr int dz = dc - 1;
                    constexpr int k = L::dir_of_code((gx + 1) * 9 + (gy + 1) * 3 + (dz + 1));
                    if constexpr (k >= 0) {
                        constexpr int sl = L::aos_slot(k);
                        f[k] = row[(sh + lz + 1 - dz) * Q + sl];
                    }
                });
            });
        } else if (cs.active) {
            load_cell<T, Q, false, LD_PULL>(a, (int)i, true, cs.mask, f);
        }
        if (cs.active) {
            collide<Q, MODEL, SHIFT>(f, a.rt);
            static_for<Q>([&](auto kc) { constexpr int sl = L::aos_slot(kc); rec[sl] = f[kc]; });
        } else {
            static_for<Q>([&](auto kc) { rec[kc] = T(0); });   // solid cells of the written array: zeros (never read)
        }
        __syncthreads();
        // the TY rows of results, each TZ*Q contiguous elements of the other array
        static_for<Q>([&](auto qc) {
            const int e = qc * (TY * TZ) + threadIdx.x;     // element of the out tile
            const int r = e / (TZ * Q), w = e - r * (TZ * Q);
            const int gy = y0 + r, gz = z0 + w / Q;
            if (gy < ny && gz < nz) a.dst[(((long long)x * ny + gy) * nz + z0) * Q + w] = out[e];
        });
        __syncthreads();   // the out tile and the buffer of layer x-1 may be reused
    }
}

}  // namespace lbm
