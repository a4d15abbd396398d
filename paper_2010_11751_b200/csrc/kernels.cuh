// kernels.cuh -- generic (one thread per cell) stream-and-collide kernels for every scheme of
// PAPER.md Table 1 (L147-159), built from three load modes and three store modes:
//
//   load   LD_LOCAL   f_k(x) = pop_k(x)                                  2-pop push, AA even, swap pass 1
//          LD_PULL    f_k(x) = pop_k(x - c_k)         | wall at x-c_k: pop_kbar(x) + w_kbar   (pull form)
//          LD_AAPULL  f_k(x) = pop_kbar(x - c_k)      | wall at x-c_k: pop_k(x)    + w_kbar   AA odd (R4)
//   store  ST_LOCAL   pop_k(x)      <- f_out_k
//          ST_SWAPPED pop_kbar(x)   <- f_out_k                           AA even, swap pass 1
//          ST_PUSH    pop_k(x+c_k)  <- f_out_k        | wall at x+c_k: pop_kbar(x) <- f_out_k + w_k
//
// with w_k = -6 t_k rho_w c_k.u_w (Eq 3; rho_w = 1, L92; zero for a resting wall).
// Instead of the paper's wall cells that store w_k in their 19 slots (Eq 4-5) a byte per
// cell says what the cell is; only fluid cells that touch a wall or the periodic seam take the
// slow path that looks at neighbour bytes, all others use fixed offsets.
//
// cell code byte: 0 = bulk fluid, 1 = wall, 2 = moving wall, 4 = fluid that needs the slow path.
#pragma once
#include "collision.cuh"

namespace lbm {

enum { LD_LOCAL = 0, LD_PULL, LD_AAPULL };
enum { ST_LOCAL = 0, ST_SWAPPED, ST_PUSH };
enum { CODE_BULK = 0, CODE_WALL = 1, CODE_MOVING = 2, CODE_EDGE = 4 };

struct Geo {
    int nx, ny, nz;
    int n;              // nx*ny*nz (< 2^31)
    long long stride;   // SoA: elements between two population planes (padded to 128 B)
};

template <class T>
struct StepArgs {
    const T* src;
    T* dst;
    const uint8_t* code;
    Geo g;
    Rates<T> rt;
    T wterm[27];  // w_k
};

template <bool SOA, int Q>
__device__ __forceinline__ long long slot(const Geo& g, int k, long long i)
{
    return SOA ? (long long)k * g.stride + i : i * Q + k;
}

__device__ __forceinline__ int wrap1(int v, int n) { return v < 0 ? v + n : (v >= n ? v - n : v); }

// index of the cell at (x + sx*cx, y + sy*cy, z + sz*cz) with periodic wrap
template <int Q, int K, int SIGN>
__device__ __forceinline__ int neighbour(const Geo& g, int x, int y, int z)
{
    using L = Lat<Q>;
    const int xx = wrap1(x + SIGN * L::cx(K), g.nx);
    const int yy = wrap1(y + SIGN * L::cy(K), g.ny);
    const int zz = wrap1(z + SIGN * L::cz(K), g.nz);
    return (xx * g.ny + yy) * g.nz + zz;
}

template <int Q, int K>
__device__ __forceinline__ int offset(const Geo& g)
{
    using L = Lat<Q>;
    return (L::cx(K) * g.ny + L::cy(K)) * g.nz + L::cz(K);
}

// ------------------------------------------------------------------ load / store of one cell
template <class T, int Q, bool SOA, int LOAD>
__device__ __forceinline__ void load_cell(const T* __restrict__ src, const uint8_t* __restrict__ code, const Geo& g,
                                          const T (&wterm)[27], int i, uint8_t mycode, T (&f)[Q])
{
    using L = Lat<Q>;
    if (LOAD == LD_LOCAL) {
        static_for<Q>([&](auto kc) { f[kc] = src[slot<SOA, Q>(g, kc, i)]; });
    } else if (mycode == CODE_BULK) {
        static_for<Q>([&](auto kc) {
            constexpr int k = kc;
            constexpr int s = LOAD == LD_PULL ? k : L::opp(k);
            f[k] = src[slot<SOA, Q>(g, s, (long long)i - offset<Q, k>(g))];
        });
    } else {
        const int z = i % g.nz, y = (i / g.nz) % g.ny, x = i / (g.nz * g.ny);
        static_for<Q>([&](auto kc) {
            constexpr int k = kc, kb = L::opp(k);
            if constexpr (k == L::REST) {
                f[k] = src[slot<SOA, Q>(g, k, i)];
            } else {
                const int n = neighbour<Q, k, -1>(g, x, y, z);
                const int nc = code[n] & 3;
                if (nc == 0) f[k] = src[slot<SOA, Q>(g, LOAD == LD_PULL ? k : kb, n)];
                else f[k] = src[slot<SOA, Q>(g, LOAD == LD_PULL ? kb : k, i)] + (nc == CODE_MOVING ? wterm[kb] : T(0));
            }
        });
    }
}

template <class T, int Q, bool SOA, int STORE>
__device__ __forceinline__ void store_cell(T* __restrict__ dst, const uint8_t* __restrict__ code, const Geo& g,
                                           const T (&wterm)[27], int i, uint8_t mycode, const T (&f)[Q])
{
    using L = Lat<Q>;
    if (STORE == ST_LOCAL) {
        static_for<Q>([&](auto kc) { dst[slot<SOA, Q>(g, kc, i)] = f[kc]; });
    } else if (STORE == ST_SWAPPED) {
        static_for<Q>([&](auto kc) { dst[slot<SOA, Q>(g, L::opp(kc), i)] = f[kc]; });
    } else if (mycode == CODE_BULK) {
        static_for<Q>([&](auto kc) {
            constexpr int k = kc;
            dst[slot<SOA, Q>(g, k, (long long)i + offset<Q, k>(g))] = f[k];
        });
    } else {
        const int z = i % g.nz, y = (i / g.nz) % g.ny, x = i / (g.nz * g.ny);
        static_for<Q>([&](auto kc) {
            constexpr int k = kc, kb = L::opp(k);
            if constexpr (k == L::REST) {
                dst[slot<SOA, Q>(g, k, i)] = f[k];
            } else {
                const int n = neighbour<Q, k, +1>(g, x, y, z);
                const int nc = code[n] & 3;
                if (nc == 0) dst[slot<SOA, Q>(g, k, n)] = f[k];
                else dst[slot<SOA, Q>(g, kb, i)] = f[k] + (nc == CODE_MOVING ? wterm[k] : T(0));
            }
        });
    }
}

// ------------------------------------------------------------------ the fused step
template <class T, int Q, int MODEL, bool SOA, int LOAD, int STORE>
__global__ void __launch_bounds__(256) step_kernel(const StepArgs<T> a)
{
    constexpr bool SHIFT = sizeof(T) == 4;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= a.g.n) return;
    const uint8_t mycode = a.code[i];
    if (mycode & 3) return;  // solid cells hold no populations
    T f[Q];
    load_cell<T, Q, SOA, LOAD>(a.src, a.code, a.g, a.wterm, i, mycode, f);
    collide<Q, MODEL, SHIFT>(f, a.rt);
    store_cell<T, Q, SOA, STORE>(a.dst, a.code, a.g, a.wterm, i, mycode, f);
}

// ------------------------------------------------------------------ swap scheme, pass 2
// After pass 1 pop_kbar(x) holds f_out_k(x).  For the half set k < NH (R5): exchange pop_kbar(x)
// with pop_k(x + c_k) when that neighbour is fluid, else add w_k in place (the value already sits
// in the slot Eq 3 sends it to); and when the neighbour at x - c_k is a wall, add w_kbar to pop_k(x).
// Every slot is touched by exactly one thread (Table 1).
template <class T, int Q, bool SOA>
__global__ void __launch_bounds__(256) swap_stream_kernel(const StepArgs<T> a)
{
    using L = Lat<Q>;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= a.g.n) return;
    const uint8_t mycode = a.code[i];
    if (mycode & 3) return;
    T* __restrict__ pop = a.dst;
    const Geo& g = a.g;
    if (mycode == CODE_BULK) {
        static_for<L::NH>([&](auto kc) {
            constexpr int k = kc, kb = L::opp(k);
            const long long pa = slot<SOA, Q>(g, kb, i);
            const long long pb = slot<SOA, Q>(g, k, (long long)i + offset<Q, k>(g));
            const T va = pop[pa], vb = pop[pb];
            pop[pa] = vb;
            pop[pb] = va;
        });
    } else {
        const int z = i % g.nz, y = (i / g.nz) % g.ny, x = i / (g.nz * g.ny);
        static_for<L::NH>([&](auto kc) {
            constexpr int k = kc, kb = L::opp(k);
            const int n = neighbour<Q, k, +1>(g, x, y, z);
            const int nc = a.code[n] & 3;
            const long long pa = slot<SOA, Q>(g, kb, i);
            if (nc == 0) {
                const long long pb = slot<SOA, Q>(g, k, n);
                const T va = pop[pa], vb = pop[pb];
                pop[pa] = vb;
                pop[pb] = va;
            } else if (nc == CODE_MOVING) {
                pop[pa] += a.wterm[k];
            }
            const int m = neighbour<Q, k, -1>(g, x, y, z);
            if ((a.code[m] & 3) == CODE_MOVING) pop[slot<SOA, Q>(g, k, i)] += a.wterm[kb];
        });
    }
}

// ------------------------------------------------------------------ set-up and exports
// model's own equilibrium on fluid cells (zero elsewhere); rho [N], u [3][N] device arrays of T
template <class T, int Q, bool EXT, bool SOA>
__global__ void init_equilibrium_kernel(T* __restrict__ pop, const uint8_t* __restrict__ code, Geo g,
                                        const T* __restrict__ rho, const T* __restrict__ u)
{
    constexpr bool SHIFT = sizeof(T) == 4;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= g.n) return;
    T E[Q];
    if (code[i] & 3) {
        static_for<Q>([&](auto kc) { E[kc] = T(0); });
    } else {
        const T r = rho[i];
        const T uu[3] = {u[i], u[(long long)g.n + i], u[2LL * g.n + i]};
        if constexpr (EXT) equilibrium_ext<Q, SHIFT>(r, uu, E);
        else equilibrium_w2<Q, SHIFT>(r, r - T(1), uu, E);
    }
    static_for<Q>([&](auto kc) { pop[slot<SOA, Q>(g, kc, i)] = E[kc]; });
}

// rho, u of the pre-collision state; LOAD says where that state lives
template <class T, int Q, bool SOA, int LOAD>
__global__ void macroscopic_kernel(const T* __restrict__ pop, const uint8_t* __restrict__ code, Geo g,
                                   StepArgs<T> a, T* __restrict__ rho, T* __restrict__ u)
{
    constexpr bool SHIFT = sizeof(T) == 4;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= g.n) return;
    const uint8_t mycode = code[i];
    T r = T(0), uu[3] = {T(0), T(0), T(0)};
    if (!(mycode & 3)) {
        T f[Q], dr;
        load_cell<T, Q, SOA, LOAD>(pop, code, g, a.wterm, i, mycode, f);
        moments_rho_u<Q, SHIFT>(f, r, dr, uu);
    }
    rho[i] = r;
    u[i] = uu[0];
    u[(long long)g.n + i] = uu[1];
    u[2LL * g.n + i] = uu[2];
}

// kinetic energy, stage 1: one double per block (fixed tree: warp shuffle, then warp 0)
template <class T, int Q, bool SOA, int LOAD>
__global__ void __launch_bounds__(256) energy_kernel(const T* __restrict__ pop, const uint8_t* __restrict__ code, Geo g,
                                                     StepArgs<T> a, double* __restrict__ partial)
{
    constexpr bool SHIFT = sizeof(T) == 4;
    double e = 0.0;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < g.n; i += (long long)gridDim.x * blockDim.x) {
        const uint8_t mycode = code[i];
        if (mycode & 3) continue;
        T f[Q], r, dr, uu[3];
        load_cell<T, Q, SOA, LOAD>(pop, code, g, a.wterm, (int)i, mycode, f);
        moments_rho_u<Q, SHIFT>(f, r, dr, uu);
        e += 0.5 * (double)r * ((double)uu[0] * uu[0] + (double)uu[1] * uu[1] + (double)uu[2] * uu[2]);
    }
    __shared__ double ws[8];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) e += __shfl_down_sync(0xffffffffu, e, o);
    if ((threadIdx.x & 31) == 0) ws[threadIdx.x >> 5] = e;
    __syncthreads();
    if (threadIdx.x < 32) {
        e = threadIdx.x < (blockDim.x >> 5) ? ws[threadIdx.x] : 0.0;
#pragma unroll
        for (int o = 4; o > 0; o >>= 1) e += __shfl_down_sync(0xffffffffu, e, o);
        if (threadIdx.x == 0) partial[blockIdx.x] = e;
    }
}

// one canonical population plane f_k(x) out of / into the internal storage.  Direction data are
// run-time here (one launch per k): source slot when the upstream cell is fluid, slot and wall
// term when it is not, and the shift (sx,sy,sz) = c_k for the pulling modes, 0 for LD_LOCAL.
struct PlaneArgs {
    int slot_fluid, slot_wall;
    int sx, sy, sz;
    double wterm;   // w_kbar
    double weight;  // t_k, added back when the storage is shifted
};
template <class T, int Q, bool SOA>
__global__ void extract_plane_kernel(const T* __restrict__ pop, const uint8_t* __restrict__ code, Geo g, PlaneArgs p,
                                     T* __restrict__ out)
{
    constexpr bool SHIFT = sizeof(T) == 4;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= g.n) return;
    T v = T(0);
    if (!(code[i] & 3)) {
        int n = i;
        if (p.sx | p.sy | p.sz) {
            const int z = i % g.nz, y = (i / g.nz) % g.ny, x = i / (g.nz * g.ny);
            n = (wrap1(x - p.sx, g.nx) * g.ny + wrap1(y - p.sy, g.ny)) * g.nz + wrap1(z - p.sz, g.nz);
        }
        const int nc = code[n] & 3;
        if (nc == 0) v = pop[slot<SOA, Q>(g, p.slot_fluid, n)];
        else v = pop[slot<SOA, Q>(g, p.slot_wall, i)] + (nc == CODE_MOVING ? T(p.wterm) : T(0));
        if (SHIFT) v += T(p.weight);
    }
    out[i] = v;
}
template <class T, int Q, bool SOA>
__global__ void insert_plane_kernel(T* __restrict__ pop, const uint8_t* __restrict__ code, Geo g, int k, double weight,
                                    const T* __restrict__ in)
{
    constexpr bool SHIFT = sizeof(T) == 4;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= g.n) return;
    T v = T(0);
    if (!(code[i] & 3)) v = SHIFT ? in[i] - T(weight) : in[i];
    pop[slot<SOA, Q>(g, k, i)] = v;
}

}  // namespace lbm
