// aux.cu -- model-independent kernels: cell classification, equilibrium initialisation, macroscopic
// export, kinetic-energy transform-reduce (reading R19),
// canonical population import/export, swap pass 2 and the stream-only pass.
#include "dispatch.cuh"

namespace lbm {

// cell code from raw flags: fluid cells on the box faces (periodic seam) or next to a non-fluid
// cell get CODE_EDGE.  The 27-neighbourhood is used for both lattices (a superset for D3Q19).
__global__ void classify_kernel(const uint8_t* __restrict__ flags, uint8_t* __restrict__ code, Geo g)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= g.n) return;
    const uint8_t fl = flags[i];
    if (fl != 0) { code[i] = fl == 2 ? CODE_MOVING : CODE_WALL; return; }
    const int z = i % g.nz, y = (i / g.nz) % g.ny, x = i / (g.nz * g.ny);
    bool edge = x == 0 || y == 0 || z == 0 || x == g.nx - 1 || y == g.ny - 1 || z == g.nz - 1;
    if (!edge) {
        for (int dx = -1; dx <= 1; ++dx)
            for (int dy = -1; dy <= 1; ++dy)
                for (int dz = -1; dz <= 1; ++dz)
                    edge |= flags[((x + dx) * g.ny + (y + dy)) * g.nz + (z + dz)] != 0;
    }
    code[i] = edge ? CODE_EDGE : CODE_BULK;
}

// energy stage 2: one block sums the per-block partials in a fixed order
__global__ void __launch_bounds__(1024) energy_final_kernel(const double* __restrict__ partial, int n, double* __restrict__ out)
{
    __shared__ double ws[32];
    double e = 0.0;
    for (int i = threadIdx.x; i < n; i += 1024) e += partial[i];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) e += __shfl_down_sync(0xffffffffu, e, o);
    if ((threadIdx.x & 31) == 0) ws[threadIdx.x >> 5] = e;
    __syncthreads();
    if (threadIdx.x < 32) {
        e = ws[threadIdx.x];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) e += __shfl_down_sync(0xffffffffu, e, o);
        if (threadIdx.x == 0) *out = e;
    }
}

// stream only: canonical f_k(x) from post-collision storage (LD_PULL), stored locally
template <class T, int Q, bool SOA>
__global__ void __launch_bounds__(256) stream_only_kernel(const StepArgs<T> a)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= a.g.n) return;
    const uint8_t mycode = a.code[i];
    if (mycode & 3) return;
    T f[Q];
    load_cell<T, Q, SOA, LD_PULL>(a.src, a.code, a.g, a.wterm, i, mycode, f);
    store_cell<T, Q, SOA, ST_LOCAL>(a.dst, a.code, a.g, a.wterm, i, mycode, f);
}

static inline int blocks_for(int n, int block) { return (n + block - 1) / block; }

cudaError_t aux_classify(const uint8_t* flags, uint8_t* code, const Geo& g, cudaStream_t s)
{
    classify_kernel<<<blocks_for(g.n, 256), 256, 0, s>>>(flags, code, g);
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
    energy_final_kernel<<<1, 1024, 0, s>>>(partial, nblocks, out);
    return cudaGetLastError();
}

template <class T>
cudaError_t aux_extract_plane(int Q, bool soa, const T* pop, const uint8_t* code, const Geo& g, const PlaneArgs& p,
                              T* out, cudaStream_t s)
{
    const int grid = blocks_for(g.n, 256);
#define CALL(QQ, SS) extract_plane_kernel<T, QQ, SS><<<grid, 256, 0, s>>>(pop, code, g, p, out)
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
    const int grid = blocks_for(a.g.n, 256);
#define CALL(QQ, SS) swap_stream_kernel<T, QQ, SS><<<grid, 256, 0, s>>>(a)
    LBM_QS_DISPATCH(Q, soa, CALL);
#undef CALL
    return cudaGetLastError();
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

#define LBM_AUX_INST(T)                                                                                                  \
    template cudaError_t aux_init_equilibrium<T>(int, bool, bool, T*, const uint8_t*, const Geo&, const T*, const T*,   \
                                                 cudaStream_t);                                                         \
    template cudaError_t aux_macroscopic<T>(int, bool, int, const StepArgs<T>&, T*, T*, cudaStream_t);                  \
    template cudaError_t aux_energy<T>(int, bool, int, const StepArgs<T>&, double*, int, double*, cudaStream_t);        \
    template cudaError_t aux_extract_plane<T>(int, bool, const T*, const uint8_t*, const Geo&, const PlaneArgs&, T*,    \
                                              cudaStream_t);                                                            \
    template cudaError_t aux_insert_plane<T>(int, bool, T*, const uint8_t*, const Geo&, int, double, const T*,          \
                                             cudaStream_t);                                                             \
    template cudaError_t aux_swap_stream<T>(int, bool, const StepArgs<T>&, cudaStream_t);                               \
    template cudaError_t aux_stream_only<T>(int, bool, const StepArgs<T>&, cudaStream_t);
LBM_AUX_INST(float)
LBM_AUX_INST(double)

template <int Q>
static void tables_of(int (*c)[3], int* opp, double* w)
{
    for (int k = 0; k < Q; ++k) {
        c[k][0] = Lat<Q>::cx(k);
        c[k][1] = Lat<Q>::cy(k);
        c[k][2] = Lat<Q>::cz(k);
        opp[k] = Lat<Q>::opp(k);
        w[k] = Lat<Q>::w(k);
    }
}
void lattice_tables(int Q, int (*c)[3], int* opp, double* w)
{
    if (Q == 19) tables_of<19>(c, opp, w);
    else tables_of<27>(c, opp, w);
}

}  // namespace lbm
