// aux.cu -- model-independent kernels: cell classification, equilibrium initialisation, macroscopic
// export, kinetic-energy transform-reduce (reading R19),
// canonical population import/export, swap pass 2 and the stream-only pass.
#include "dispatch.cuh"

namespace lbm {

// cell code and link mask (kernels.cuh) from raw flags.  A fluid cell gets CODE_EDGE when its
// mask is non-zero: a link of the lattice ends on a non-fluid cell, or the cell lies on a face of
// the box (periodic seam).
template <int Q>
__device__ __forceinline__ unsigned long long link_mask(const uint8_t* __restrict__ flags, const Geo& g, int i)
{
    using L = Lat<Q>;
    const int z = i % g.nz, y = (i / g.nz) % g.ny, x = i / (g.nz * g.ny);
    unsigned long long m = 0ull;
    if (x == 0) m |= 1ull << (MASK_FACE_SHIFT + 0);
    if (x == g.nx - 1) m |= 1ull << (MASK_FACE_SHIFT + 1);
    if (y == 0) m |= 1ull << (MASK_FACE_SHIFT + 2);
    if (y == g.ny - 1) m |= 1ull << (MASK_FACE_SHIFT + 3);
    if (z == 0) m |= 1ull << (MASK_FACE_SHIFT + 4);
    if (z == g.nz - 1) m |= 1ull << (MASK_FACE_SHIFT + 5);
    static_for<Q>([&](auto kc) {
        constexpr int k = kc;
        if constexpr (k != L::REST) {
            const int n = (wrap1(x + L::cx(k), g.nx) * g.ny + wrap1(y + L::cy(k), g.ny)) * g.nz + wrap1(z + L::cz(k), g.nz);
            const uint8_t nf = flags[n];
            if (nf == 1 || nf == 2) m |= 1ull << link_of<Q>(k);  // a ghost neighbour (3) is read like a fluid one
            if (nf == 2) m |= 1ull << (MASK_MOVING_SHIFT + link_of<Q>(k));
        }
    });
    return m;
}

// pass 1: the code byte of every cell and, per aligned group of 32 cells (one warp), the bit set of
// its edge cells (grp.y) and their number (grp.x, turned into an exclusive prefix sum by pass 2)
template <int Q>
__global__ void __launch_bounds__(256) classify_kernel(const uint8_t* __restrict__ flags, uint8_t* __restrict__ code,
                                                        uint2* __restrict__ grp, Geo g)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    bool edge = false;
    if (i < g.n) {
        const uint8_t fl = flags[i];
        uint8_t c;
        if (fl != 0) c = fl == 2 ? CODE_MOVING : fl == 3 ? CODE_GHOST : CODE_WALL;
        else { edge = link_mask<Q>(flags, g, i) != 0ull; c = edge ? CODE_EDGE : CODE_BULK; }
        code[i] = c;
    }
    const unsigned bits = __ballot_sync(0xffffffffu, edge);
    if ((threadIdx.x & 31) == 0 && i < g.n) grp[i >> 5] = make_uint2((unsigned)__popc(bits), bits);
}

// pass 2: exclusive prefix sum of grp[].x over the ngrp groups, in three launches: per block of 1024
// groups its sum (sums[b]); one block turns sums[] into exclusive prefixes and leaves the grand total
// (the number of edge cells) in total[0]; every block then scans its own 1024 entries from its prefix
__device__ __forceinline__ unsigned block_scan_1024(unsigned v, unsigned* warp_tot)
{
    // inclusive scan over the 1024 threads of the block; warp_tot: 32 unsigned of shared memory
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const unsigned t = __shfl_up_sync(0xffffffffu, v, o);
        if (lane >= o) v += t;
    }
    if (lane == 31) warp_tot[w] = v;
    __syncthreads();
    if (w == 0) {
        unsigned t = warp_tot[lane];
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const unsigned u = __shfl_up_sync(0xffffffffu, t, o);
            if (lane >= o) t += u;
        }
        warp_tot[lane] = t;
    }
    __syncthreads();
    if (w > 0) v += warp_tot[w - 1];
    return v;
}
__global__ void __launch_bounds__(1024) classify_sum_kernel(const uint2* __restrict__ grp, int ngrp, unsigned* __restrict__ sums)
{
    __shared__ unsigned wt[32];
    const int j = blockIdx.x * 1024 + threadIdx.x;
    const unsigned v = block_scan_1024(j < ngrp ? grp[j].x : 0u, wt);
    if (threadIdx.x == 1023) sums[blockIdx.x] = v;
}
__global__ void __launch_bounds__(1024) classify_scan_sums_kernel(unsigned* __restrict__ sums, int nb, unsigned* __restrict__ total)
{
    __shared__ unsigned wt[32];
    __shared__ unsigned carry;
    if (threadIdx.x == 0) carry = 0u;
    __syncthreads();
    for (int base = 0; base < nb; base += 1024) {
        const int j = base + threadIdx.x;
        const unsigned mine = j < nb ? sums[j] : 0u;
        const unsigned incl = block_scan_1024(mine, wt);
        const unsigned c = carry;
        if (j < nb) sums[j] = c + incl - mine;
        __syncthreads();
        if (threadIdx.x == 1023) carry = c + incl;
        __syncthreads();
    }
    if (threadIdx.x == 0) total[0] = carry;
}
__global__ void __launch_bounds__(1024) classify_apply_kernel(uint2* __restrict__ grp, int ngrp, const unsigned* __restrict__ sums)
{
    __shared__ unsigned wt[32];
    const int j = blockIdx.x * 1024 + threadIdx.x;
    const unsigned mine = j < ngrp ? grp[j].x : 0u;
    const unsigned incl = block_scan_1024(mine, wt);
    if (j < ngrp) grp[j].x = sums[blockIdx.x] + incl - mine;
}

// pass 3: the masks of the edge cells, in cell order
template <int Q>
__global__ void __launch_bounds__(256) classify_mask_kernel(const uint8_t* __restrict__ flags, const uint8_t* __restrict__ code,
                                                             const uint2* __restrict__ grp, unsigned long long* __restrict__ mask, Geo g)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= g.n || code[i] != CODE_EDGE) return;
    const uint2 gg = grp[i >> 5];
    mask[gg.x + __popc(gg.y & ((1u << (i & 31)) - 1u))] = link_mask<Q>(flags, g, i);
}

// energy stages 2 and 3: block b sums the contiguous segment [b*seg, min(n, (b+1)*seg)) of `in` in a
// fixed order into out[b]; launched once with many blocks and once with a single block
__global__ void __launch_bounds__(256) energy_sum_kernel(const double* __restrict__ in, int n, int seg, double* __restrict__ out)
{
    __shared__ double ws[8];
    const int lo = blockIdx.x * seg, hi = min(n, lo + seg);
    double e = 0.0;
    for (int i = lo + threadIdx.x; i < hi; i += 256) e += in[i];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) e += __shfl_down_sync(0xffffffffu, e, o);
    if ((threadIdx.x & 31) == 0) ws[threadIdx.x >> 5] = e;
    __syncthreads();
    if (threadIdx.x < 32) {
        e = threadIdx.x < 8 ? ws[threadIdx.x] : 0.0;
#pragma unroll
        for (int o = 4; o > 0; o >>= 1) e += __shfl_down_sync(0xffffffffu, e, o);
        if (threadIdx.x == 0) out[blockIdx.x] = e;
    }
}

// stream only: canonical f_k(x) from post-collision storage (LD_PULL), stored locally
template <class T, int Q, bool SOA>
__global__ void __launch_bounds__(256) stream_only_kernel(const StepArgs<T> a)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const CellState cs = cell_state(a, i, a.g.n);
    if (!cs.active) return;
    T f[Q];
    load_cell<T, Q, SOA, LD_PULL>(a, i, cs.masked, cs.mask, f);
    store_cell<T, Q, SOA, ST_LOCAL>(a, i, cs.masked, cs.mask, f);
}

static inline int blocks_for(int n, int block) { return (n + block - 1) / block; }

// sums: scratch of ceil(ngrp / 1024) unsigned, ngrp = ceil(n / 32)
cudaError_t aux_classify_codes(int Q, const uint8_t* flags, uint8_t* code, uint2* grp, unsigned* total, unsigned* sums,
                               const Geo& g, cudaStream_t s)
{
    if (Q == 19) classify_kernel<19><<<blocks_for(g.n, 256), 256, 0, s>>>(flags, code, grp, g);
    else if (Q == 27) classify_kernel<27><<<blocks_for(g.n, 256), 256, 0, s>>>(flags, code, grp, g);
    else return cudaErrorInvalidValue;
    const int ngrp = (g.n + 31) / 32, nb = (ngrp + 1023) / 1024;
    classify_sum_kernel<<<nb, 1024, 0, s>>>(grp, ngrp, sums);
    classify_scan_sums_kernel<<<1, 1024, 0, s>>>(sums, nb, total);
    classify_apply_kernel<<<nb, 1024, 0, s>>>(grp, ngrp, sums);
    return cudaGetLastError();
}
cudaError_t aux_classify_masks(int Q, const uint8_t* flags, const uint8_t* code, const uint2* grp, unsigned long long* mask,
                               const Geo& g, cudaStream_t s)
{
    if (Q == 19) classify_mask_kernel<19><<<blocks_for(g.n, 256), 256, 0, s>>>(flags, code, grp, mask, g);
    else if (Q == 27) classify_mask_kernel<27><<<blocks_for(g.n, 256), 256, 0, s>>>(flags, code, grp, mask, g);
    else return cudaErrorInvalidValue;
    return cudaGetLastError();
}

// run-time (Q, soa) -> compile-time
#define LBM_QS_DISPATCH(Q, soa, CALL)                   \
    do {                                                \
        if ((Q) == 19 && (soa)) { CALL(19, true); }     \
        else if ((Q) == 19) { CALL(19, false); }        \
        else if ((Q) == 27 && (soa)) { CALL(27, true); } \
        else if ((Q) == 27) { CALL(27, false); }        \
        else return cudaErrorInvalidValue;              \
    } while (0)

template <class T>
cudaError_t aux_init_equilibrium(int Q, bool ext, bool soa, T* pop, const uint8_t* code, const Geo& g, const T* rho,
                                 const T* u, cudaStream_t s)
{
    const int grid = blocks_for(g.n, 128);
#define CALL(QQ, SS)                                                                              \
    if (ext) init_equilibrium_kernel<T, QQ, true, SS><<<grid, 128, 0, s>>>(pop, code, g, rho, u); \
    else init_equilibrium_kernel<T, QQ, false, SS><<<grid, 128, 0, s>>>(pop, code, g, rho, u)
    LBM_QS_DISPATCH(Q, soa, CALL);
#undef CALL
    return cudaGetLastError();
}

template <class T>
cudaError_t aux_macroscopic(int Q, bool soa, int load, const StepArgs<T>& a, T* rho, T* u, cudaStream_t s)
{
    const int grid = blocks_for(a.g.n, 256);
#define CALL(QQ, SS)                                                                                              \
    switch (load) {                                                                                               \
    case LD_LOCAL: macroscopic_kernel<T, QQ, SS, LD_LOCAL><<<grid, 256, 0, s>>>(a.src, a.code, a.g, a, rho, u); break;   \
    case LD_PULL: macroscopic_kernel<T, QQ, SS, LD_PULL><<<grid, 256, 0, s>>>(a.src, a.code, a.g, a, rho, u); break;     \
    case LD_AAPULL: macroscopic_kernel<T, QQ, SS, LD_AAPULL><<<grid, 256, 0, s>>>(a.src, a.code, a.g, a, rho, u); break; \
    default: return cudaErrorInvalidValue;                                                                        \
    }
    LBM_QS_DISPATCH(Q, soa, CALL);
#undef CALL
    return cudaGetLastError();
}

// partial: [nblocks + ENERGY_STAGE2] doubles, nblocks = ceil(n / 256); out: one double
template <class T>
cudaError_t aux_energy(int Q, bool soa, int load, const StepArgs<T>& a, double* partial, int nblocks, double* out,
                       cudaStream_t s)
{
#define CALL(QQ, SS)                                                                                                \
    switch (load) {                                                                                                 \
    case LD_LOCAL: energy_kernel<T, QQ, SS, LD_LOCAL><<<nblocks, 256, 0, s>>>(a.src, a.code, a.g, a, partial); break;     \
    case LD_PULL: energy_kernel<T, QQ, SS, LD_PULL><<<nblocks, 256, 0, s>>>(a.src, a.code, a.g, a, partial); break;       \
    case LD_AAPULL: energy_kernel<T, QQ, SS, LD_AAPULL><<<nblocks, 256, 0, s>>>(a.src, a.code, a.g, a, partial); break;   \
    default: return cudaErrorInvalidValue;                                                                          \
    }
    LBM_QS_DISPATCH(Q, soa, CALL);
#undef CALL
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    const int seg = (nblocks + ENERGY_STAGE2 - 1) / ENERGY_STAGE2;
    const int n2 = (nblocks + seg - 1) / seg;
    energy_sum_kernel<<<n2, 256, 0, s>>>(partial, nblocks, seg, partial + nblocks);
    energy_sum_kernel<<<1, 256, 0, s>>>(partial + nblocks, n2, n2, out);
    return cudaGetLastError();
}

template <class T>
cudaError_t aux_extract_plane(int Q, bool soa, const T* pop, const uint8_t* code, const Geo& g, const PlaneArgs& p,
                              T* out, const int* cells, int m, cudaStream_t s)
{
    const int grid = blocks_for(m, 256);
#define CALL(QQ, SS) extract_plane_kernel<T, QQ, SS><<<grid, 256, 0, s>>>(pop, code, g, p, out, cells, m)
    LBM_QS_DISPATCH(Q, soa, CALL);
#undef CALL
    return cudaGetLastError();
}

template <class T>
cudaError_t aux_insert_plane(int Q, bool soa, T* pop, const uint8_t* code, const Geo& g, int k, double weight,
                             const T* in, cudaStream_t s)
{
    const int grid = blocks_for(g.n, 256);
#define CALL(QQ, SS) insert_plane_kernel<T, QQ, SS><<<grid, 256, 0, s>>>(pop, code, g, k, weight, in)
    LBM_QS_DISPATCH(Q, soa, CALL);
#undef CALL
    return cudaGetLastError();
}

template <class T>
cudaError_t aux_swap_stream(int Q, bool soa, const StepArgs<T>& a, cudaStream_t s)
{
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cudaLaunchConfig_t cfg = {};
    cfg.stream = s;
    cfg.attrs = attr;
    cfg.numAttrs = a.pdl ? 1 : 0;
    cudaError_t e = cudaSuccess;
    if (!soa) {   // AoS: cooperative exchange of the slot triples (kernels.cuh)
        const int grid = blocks_for(a.g.n, 128);
        const size_t smem = (size_t)(128 / 32) * 192 * sizeof(T);
        if (Q == 19) swap_stream_kernel_aos<T, 19><<<grid, 128, smem, s>>>(a);
        else if (Q == 27) swap_stream_kernel_aos<T, 27><<<grid, 128, smem, s>>>(a);
        else return cudaErrorInvalidValue;
        return cudaGetLastError();
    }
#define CALL(QQ, SS)                                                                   \
    {                                                                                  \
        constexpr int G = swap_groups<T, QQ>();                                        \
        constexpr int b = G > 1 ? 256 : (swap_max_threads<T, QQ>() < 256 ? swap_max_threads<T, QQ>() : 256); \
        cfg.gridDim = dim3(blocks_for(a.g.n, b), G);                                   \
        cfg.blockDim = dim3(b);                                                        \
        e = cudaLaunchKernelEx(&cfg, swap_stream_kernel<T, QQ, SS, G>, a);             \
    }
    LBM_QS_DISPATCH(Q, soa, CALL);
#undef CALL
    return e;
}

template <class T>
cudaError_t aux_stream_only(int Q, bool soa, const StepArgs<T>& a, cudaStream_t s)
{
    const int grid = blocks_for(a.g.n, 256);
#define CALL(QQ, SS) stream_only_kernel<T, QQ, SS><<<grid, 256, 0, s>>>(a)
    LBM_QS_DISPATCH(Q, soa, CALL);
#undef CALL
    return cudaGetLastError();
}

template <class T>
cudaError_t aux_halo(bool pack, T* pop, const uint8_t* code, long long stride, const HaloArgs& p, T* buf, cudaStream_t s)
{
    const dim3 grid((p.cells + 255) / 256, p.ndir);
    if (pack) halo_kernel<T, true><<<grid, 256, 0, s>>>(pop, code, stride, p, buf);
    else halo_kernel<T, false><<<grid, 256, 0, s>>>(pop, code, stride, p, buf);
    return cudaGetLastError();
}

#define LBM_AUX_INST(T)                                                                                                  \
    template cudaError_t aux_init_equilibrium<T>(int, bool, bool, T*, const uint8_t*, const Geo&, const T*, const T*,   \
                                                 cudaStream_t);                                                         \
    template cudaError_t aux_macroscopic<T>(int, bool, int, const StepArgs<T>&, T*, T*, cudaStream_t);                  \
    template cudaError_t aux_energy<T>(int, bool, int, const StepArgs<T>&, double*, int, double*, cudaStream_t);        \
    template cudaError_t aux_extract_plane<T>(int, bool, const T*, const uint8_t*, const Geo&, const PlaneArgs&, T*,    \
                                              const int*, int, cudaStream_t);                                                           \
    template cudaError_t aux_insert_plane<T>(int, bool, T*, const uint8_t*, const Geo&, int, double, const T*,          \
                                             cudaStream_t);                                                             \
    template cudaError_t aux_halo<T>(bool, T*, const uint8_t*, long long, const HaloArgs&, T*, cudaStream_t);                           \
    template cudaError_t aux_swap_stream<T>(int, bool, const StepArgs<T>&, cudaStream_t);                               \
    template cudaError_t aux_stream_only<T>(int, bool, const StepArgs<T>&, cudaStream_t);
LBM_AUX_INST(float)
LBM_AUX_INST(double)

template <int Q>
static void tables_of(int (*c)[3], int* opp, double* w, int* aos)
{
    for (int k = 0; k < Q; ++k) {
        aos[k] = Lat<Q>::aos_slot(k);
        c[k][0] = Lat<Q>::cx(k);
        c[k][1] = Lat<Q>::cy(k);
        c[k][2] = Lat<Q>::cz(k);
        opp[k] = Lat<Q>::opp(k);
        w[k] = Lat<Q>::w(k);
    }
}
void lattice_tables(int Q, int (*c)[3], int* opp, double* w, int* aos)
{
    if (Q == 19) tables_of<19>(c, opp, w, aos);
    else tables_of<27>(c, opp, w, aos);
}

}  // namespace lbm
