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
// cell says what the cell is, and fluid cells that touch a non-fluid cell or a face of the box
// carry a 64-bit link mask (built once by classify_kernel):
//
//   bits  0..25  link l: the neighbour at x + c_k is not fluid            (l = k, rest skipped)
//   bits 26..51  link l: that neighbour is a MOVING wall
//   bits 52..57  the cell lies on the face x=0, x=nx-1, y=0, y=ny-1, z=0, z=nz-1 (periodic seam)
//
// The masks are stored compactly, one per EDGE cell in cell order (a 512^3 cavity has 1.6 M of them,
// not 134 M): `grp[i >> 5]` holds, per aligned group of 32 cells, the ordinal of the group's first
// edge cell (x) and the bit set of its edge cells (y), so that the mask of edge cell i is
// mask[grp.x + popc(grp.y & lanes below i)].  Side arrays: 1 B (code) + 0.25 B (grp) per cell.
//
// A warp in which no lane has a mask runs the pure path (fixed offsets, no tests); a warp with at
// least one masked lane runs the masked path for all its lanes (selects on mask bits, no
// divergence, no integer division).  Both give the same values for bulk cells.
//
// cell code byte: 0 = bulk fluid, 1 = wall, 2 = moving wall, 3 = ghost (a fluid cell that another
// rank owns: never updated here, read like a fluid cell by its neighbours, filled by
// halo_unpack), 4 = fluid with a non-zero link mask.
#pragma once
#include "collision.cuh"

namespace lbm {

enum { LD_LOCAL = 0, LD_PULL, LD_AAPULL };
enum { ST_LOCAL = 0, ST_SWAPPED, ST_PUSH };
enum { CODE_BULK = 0, CODE_WALL = 1, CODE_MOVING = 2, CODE_GHOST = 3, CODE_EDGE = 4 };
enum { MASK_MOVING_SHIFT = 26, MASK_FACE_SHIFT = 52 };

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
    const uint2* grp;                  // per 32 cells: ordinal of the first edge cell, bit set of edge cells
    const unsigned long long* mask;    // link masks of the edge cells, in cell order
    Geo g;
    int first, end;   // the step kernel updates the cells [first, end): the whole box, or some x-layers (slab overlap)
    int pdl;          // host side: launch with programmatic stream serialisation (see step_kernel)
    int pf;           // L2 prefetch distance in cells (0 = off), see step_kernel
    int pf_strided;   // one warp in 128/sizeof(T) prefetches, each lane a different line
    int tma;          // host side: run step_kernel_tma (tma_step.cuh) when the launch allows it
    int march;        // host side: AoS two-population pull may run step_kernel_aos_march (outer x-layers solid)
    int patch;        // host side: AoS two-population pull runs step_kernel_aos_pull_patch (the default)
    int rev;          // the blocks of step_kernel / swap_stream_kernel walk the cells from the top down
    Rates<T> rt;
    T wterm[27];  // w_k
    // offsets filled on the host per launch (make_args) so that the kernels add one uniform
    // 64-bit constant per direction instead of multiplying strides per thread:
    //   plane[k]  slot k of cell 0, in elements          (SoA: k*stride, AoS: k)
    //   ldo[k]    where the pure load of f_k starts, in BYTES: LD_LOCAL plane[k]; LD_PULL
    //             plane[k] - off_k*IS; LD_AAPULL plane[kbar] - off_k*IS   (times sizeof(T))
    //   sto[k]    where the pure store of f_k goes, in BYTES: ST_LOCAL plane[k]; ST_SWAPPED
    //             plane[kbar]; ST_PUSH plane[k] + off_k*IS                (times sizeof(T))
    // with IS = 1 (SoA) or Q (AoS) elements per cell step and off_k the cell-index offset of c_k.
    //   wlo[k]    byte offset of the slot the masked load of f_k reads when the upstream cell is
    //             solid: LD_PULL plane[kbar]; LD_AAPULL plane[k]
    //   wso[k]    byte offset of the slot the masked ST_PUSH store of f_k writes when the
    //             downstream cell is solid: plane[kbar]
    long long plane[27], ldo[27], sto[27], wlo[27], wso[27];
    // SoA: the same as pointers, lp[k] = src + ldo[k], sp[k] = dst + sto[k] (in elements), so that the
    // pure access of cell i is lp[k][i] with a 32-bit i: one IMAD.WIDE with the pointer taken from the
    // constant bank instead of a 64-bit add in two instructions (57 fewer integer instructions per
    // D3Q19 cell: the fp32 kernels are close to issue-bound)
    const T* lp[27];
    T* sp[27];
};

// element index of STORAGE slot s of cell i (SoA: plane s; AoS: s-th value of the record)
template <bool SOA, int Q>
__device__ __forceinline__ long long slot_raw(const Geo& g, int s, long long i)
{
    return SOA ? (long long)s * g.stride + i : i * Q + s;
}
// storage slot of direction K: K itself in SoA, Lat<Q>::aos_slot(K) in AoS
template <bool SOA, int Q, int K>
__host__ __device__ constexpr int storage_slot()
{
    return SOA ? K : Lat<Q>::aos_slot(K);
}
// element index of direction K (compile-time) of cell i
template <bool SOA, int Q, int K>
__device__ __forceinline__ long long slot(const Geo& g, long long i)
{
    constexpr int s = storage_slot<SOA, Q, K>();
    return slot_raw<SOA, Q>(g, s, i);
}

__device__ __forceinline__ int wrap1(int v, int n) { return v < 0 ? v + n : (v >= n ? v - n : v); }

template <int Q, int K>
__device__ __forceinline__ int offset(const Geo& g)
{
    using L = Lat<Q>;
    return (L::cx(K) * g.ny + L::cy(K)) * g.nz + L::cz(K);
}

// link index of direction k in the mask (the rest velocity has no link)
template <int Q>
__host__ __device__ constexpr int link_of(int k) { return k < Lat<Q>::REST ? k : k - 1; }

// per-thread view of a link mask
struct Edge {
    unsigned solid, moving, face;
    // cell-index corrections that turn the plain neighbour offset into the periodically wrapped one
    // (zero unless the cell lies on that face of the box)
    int fxm, fxp, fym, fyp, fzm, fzp;
    __device__ __forceinline__ Edge(unsigned long long mask, const Geo& g)
    {
        solid = (unsigned)mask & ((1u << MASK_MOVING_SHIFT) - 1u);
        moving = (unsigned)(mask >> MASK_MOVING_SHIFT) & ((1u << MASK_MOVING_SHIFT) - 1u);
        face = (unsigned)(mask >> MASK_FACE_SHIFT);
        const int sx = g.ny * g.nz, sy = g.nz;
        fxm = (face & 1u) ? g.nx * sx : 0;
        fxp = (face & 2u) ? -g.nx * sx : 0;
        fym = (face & 4u) ? g.ny * sy : 0;
        fyp = (face & 8u) ? -g.ny * sy : 0;
        fzm = (face & 16u) ? g.nz : 0;
        fzp = (face & 32u) ? -g.nz : 0;
    }
    // wrap correction (in cells) of the neighbour at x + SIGN * c_K
    template <int Q, int K, int SIGN>
    __device__ __forceinline__ int fix() const
    {
        using L = Lat<Q>;
        constexpr int dx = SIGN * L::cx(K), dy = SIGN * L::cy(K), dz = SIGN * L::cz(K);
        int o = 0;
        if constexpr (dx == 1) o += fxp;
        if constexpr (dx == -1) o += fxm;
        if constexpr (dy == 1) o += fyp;
        if constexpr (dy == -1) o += fym;
        if constexpr (dz == 1) o += fzp;
        if constexpr (dz == -1) o += fzm;
        return o;
    }
    // index offset to the cell at x + SIGN * c_K, periodic wrap included
    template <int Q, int K, int SIGN>
    __device__ __forceinline__ int off(const Geo& g) const
    {
        return SIGN * offset<Q, K>(g) + fix<Q, K, SIGN>();
    }
    template <int Q, int K>
    __device__ __forceinline__ bool solid_at() const { return (solid >> link_of<Q>(K)) & 1u; }
    template <int Q, int K>
    __device__ __forceinline__ bool moving_at() const { return (moving >> link_of<Q>(K)) & 1u; }
};

// ------------------------------------------------------------------ load / store of one cell
// `masked` must be warp-uniform; mask is this cell's link mask (0 for a bulk cell)
template <class T, int Q, bool SOA, int LOAD>
__device__ __forceinline__ void load_cell(const StepArgs<T>& a, int i, bool masked, unsigned long long mask, T (&f)[Q])
{
    using L = Lat<Q>;
    constexpr int IS = SOA ? 1 : Q;
    const T* __restrict__ src = a.src;
    if (LOAD == LD_LOCAL || !masked) {
        if constexpr (SOA) {
            static_for<Q>([&](auto kc) { f[kc] = a.lp[kc][i]; });
        } else {
            const char* __restrict__ p = reinterpret_cast<const char*>(src + (long long)i * IS);
            static_for<Q>([&](auto kc) { f[kc] = *reinterpret_cast<const T*>(p + a.ldo[kc]); });
        }
    } else {
        const Edge e(mask, a.g);
        const char* __restrict__ p = reinterpret_cast<const char*>(src + (long long)i * IS);
        // FACES: some lane of the (converged part of the) warp lies on a face of the box and needs the
        // periodic wrap corrections.  In a cavity or a channel no fluid cell does -- the masked warps
        // are the ones next to walls -- and the corrections (up to three adds per link) are skipped.
        auto body = [&](auto faces) {
            static_for<Q>([&](auto kc) {
                constexpr int k = kc, kb = L::opp(k);
                if constexpr (k == L::REST) {
                    f[k] = *reinterpret_cast<const T*>(p + a.ldo[k]);
                } else {
                    // the upstream neighbour x - c_k = x + c_kbar: link kbar
                    long long o_fluid = a.ldo[k];
                    if constexpr (decltype(faces)::value) o_fluid += (long long)e.template fix<Q, k, -1>() * (long long)(IS * sizeof(T));
                    T v = *reinterpret_cast<const T*>(p + (e.template solid_at<Q, kb>() ? a.wlo[k] : o_fluid));
                    if (e.template moving_at<Q, kb>()) v += a.wterm[kb];
                    f[k] = v;
                }
            });
        };
        if (__any_sync(__activemask(), e.face != 0u)) body(IC<1>{});
        else body(IC<0>{});
    }
}

template <class T, int Q, bool SOA, int STORE>
__device__ __forceinline__ void store_cell(const StepArgs<T>& a, int i, bool masked, unsigned long long mask, const T (&f)[Q])
{
    using L = Lat<Q>;
    constexpr int IS = SOA ? 1 : Q;
    T* __restrict__ dst = a.dst;
    if (STORE != ST_PUSH || !masked) {
        if constexpr (SOA) {
            static_for<Q>([&](auto kc) { a.sp[kc][i] = f[kc]; });
        } else {
            char* __restrict__ p = reinterpret_cast<char*>(dst + (long long)i * IS);
            static_for<Q>([&](auto kc) { *reinterpret_cast<T*>(p + a.sto[kc]) = f[kc]; });
        }
    } else {
        const Edge e(mask, a.g);
        char* __restrict__ p = reinterpret_cast<char*>(dst + (long long)i * IS);
        auto body = [&](auto faces) {   // see load_cell
            static_for<Q>([&](auto kc) {
                constexpr int k = kc;
                if constexpr (k == L::REST) {
                    *reinterpret_cast<T*>(p + a.sto[k]) = f[k];
                } else {
                    long long o_fluid = a.sto[k];
                    if constexpr (decltype(faces)::value) o_fluid += (long long)e.template fix<Q, k, +1>() * (long long)(IS * sizeof(T));
                    T v = f[k];
                    if (e.template moving_at<Q, k>()) v += a.wterm[k];
                    *reinterpret_cast<T*>(p + (e.template solid_at<Q, k>() ? a.wso[k] : o_fluid)) = v;
                }
            });
        };
        if (__any_sync(__activemask(), e.face != 0u)) body(IC<1>{});
        else body(IC<0>{});
    }
}

// what every cell kernel starts with: is this thread's cell fluid, and does its warp need masks
struct CellState {
    bool active, masked;
    bool partial;   // inactive lane of a warp that has active lanes
    unsigned long long mask;
};
__device__ __forceinline__ unsigned long long edge_mask(const uint2* __restrict__ grp,
                                                        const unsigned long long* __restrict__ mask, long long i)
{
    const uint2 g = grp[i >> 5];
    return mask[g.x + __popc(g.y & ((1u << (i & 31)) - 1u))];
}
// EAGER: the group-table entry is fetched alongside the code byte (one sector per warp), so that the mask
// of an edge cell is one dependent load away instead of two; costs two registers, which swap pass 2 at
// its 48-register cap does not have (D3Q27 fp64: 136 -> 156 bytes of spills, 93.9 -> 91.0 %)
template <bool EAGER = true, class ARGS>
__device__ __forceinline__ CellState cell_state(const ARGS& a, long long i, int n)
{
    CellState s;
    uint8_t c = CODE_WALL;
    uint2 g = make_uint2(0u, 0u);
    if (i < n) {
        c = a.code[i];
        if constexpr (EAGER) g = a.grp[i >> 5];
    }
    s.active = !(c & 3);
    const bool edge = c == CODE_EDGE;
    s.masked = __any_sync(0xffffffffu, edge);
    const bool any_active = __any_sync(0xffffffffu, s.active);
    s.partial = any_active && !s.active && i < n;
    if constexpr (EAGER) s.mask = edge ? a.mask[g.x + __popc(g.y & ((1u << (i & 31)) - 1u))] : 0ull;
    else s.mask = edge ? edge_mask(a.grp, a.mask, i) : 0ull;
    return s;
}

// ------------------------------------------------------------------ the fused step
// __launch_bounds__(max_threads, min_blocks) = the register cap 65536 / (max_threads * min_blocks),
// tuned on B200 per precision and lattice: fp64 D3Q19 128 x 7 (72 registers, 28 warps per SM), fp64
// D3Q27 128 x 5 (96 registers: 20 warps per SM instead of the 16 that 128 registers allow), fp32 D3Q19 256 x 6 (40), fp32
// D3Q27 256 x 5 (48; round 2: 256 x 4 = 64 registers was 1-3 points slower for every model in the AA scheme).  Launches clamp the block size to max_threads.
#ifndef LBM_MINB_D19
#define LBM_MINB_D19 7
#endif
#ifndef LBM_MAXT_D27
#define LBM_MAXT_D27 128
#endif
#ifndef LBM_MINB_D27
#define LBM_MINB_D27 5
#endif
#ifndef LBM_MINB_F
#define LBM_MINB_F 6
#endif
#ifndef LBM_MINB_F27
#define LBM_MINB_F27 5
#endif
template <class T, int Q>
constexpr int min_blocks() { return sizeof(T) == 4 ? (Q == 19 ? LBM_MINB_F : LBM_MINB_F27) : Q == 19 ? LBM_MINB_D19 : LBM_MINB_D27; }
#ifndef LBM_MAXT_D19
#define LBM_MAXT_D19 128
#endif
#ifndef LBM_MAXT_F
#define LBM_MAXT_F 256
#endif
#ifndef LBM_MAXT_F27
#define LBM_MAXT_F27 256
#endif
template <class T, int Q>
constexpr int max_threads() { return sizeof(T) == 4 ? (Q == 19 ? LBM_MAXT_F : LBM_MAXT_F27) : Q == 19 ? LBM_MAXT_D19 : LBM_MAXT_D27; }

template <class T, int Q, int MODEL, bool SOA, int LOAD, int STORE>
__global__ void __launch_bounds__(max_threads<T, Q>(), min_blocks<T, Q>()) step_kernel(const StepArgs<T> a)
{
    constexpr bool SHIFT = sizeof(T) == 4;
    // Programmatic dependent launch: the next step kernel of the stream may be scheduled as soon as
    // every block of this one has started, and runs its prologue (cell codes and link masks, which
    // no step kernel writes) while this grid drains; it touches populations only after
    // griddepcontrol.wait, i.e. once this grid has completed and its stores are visible.  Without
    // the launch attribute both instructions do nothing.
    asm volatile("griddepcontrol.launch_dependents;");
    // a.rev: the blocks walk the cells from the top down.  Successive step kernels alternate the direction
    // (host: step_kind), so each starts on the ~100 MB of lines its predecessor touched last, which are still
    // in the 126 MB L2: those reads hit, and in the in-place schemes the lines are overwritten there before
    // they were ever written back.  Less DRAM traffic than the algorithmic bytes; nothing for the arithmetic.
    const unsigned blk = a.rev ? gridDim.x - 1u - blockIdx.x : blockIdx.x;
    const int i = a.first + blk * blockDim.x + threadIdx.x;
    const CellState cs = cell_state(a, i, a.end);
    asm volatile("griddepcontrol.wait;" ::: "memory");
    if (!cs.active) {  // solid cells hold no populations
        // ... but when the other array is written (two-population), a warp that straddles a wall
        // fills the wall cells' slots too: a partially written 32 B sector that is not in L2 costs
        // a DRAM read-modify-write when it is evicted (ncu: +80 MB read per 256^3 step, both precisions)
        if constexpr (STORE == ST_LOCAL && LOAD != LD_LOCAL) {
            if (cs.partial) {
                if constexpr (SOA) {
                    static_for<Q>([&](auto kc) { a.sp[kc][i] = T(0); });
                } else {
                    char* __restrict__ p = reinterpret_cast<char*>(a.dst + (long long)i * Q);
                    static_for<Q>([&](auto kc) { *reinterpret_cast<T*>(p + a.sto[kc]) = T(0); });
                }
            }
        }
        return;
    }
    // The loads in flight of a step kernel live in registers (one cell per thread), and the register
    // file caps them below what hides the DRAM latency at full bandwidth (fp32 worst: 4 bytes per
    // destination register).  So the kernel also asks L2 for the lines of the cells `pf` cells
    // ahead: no registers held, and the blocks scheduled next find their loads in L2.  fp64: every
    // thread prefetches for the cell pf ahead of its own (16384 cells; 2048 ... 32768 do equally).
    // fp32 cannot afford Q more instructions per thread (the pull kernel loses 15 % that way), so
    // one warp in 32 prefetches with each lane on a different 128 B line: 32 lines = the next 1024
    // cells of each plane (65536 cells ahead).  Measured, same box, prefetch off -> on: AA fp32
    // 88.0 -> 95.2 %, 2-pop fp32 86.7 -> 90.6 %, cumulants AA fp32 82.7 -> 89.1 %, AA fp64 98.9 ->
    // 100.5 %, D3Q27 cumulants AA fp64 92.0 -> 96.2 %, 128^3 AA fp64 94.0 -> 95.9 %.
    if (a.pf != 0) {   // negative: the cells behind, for a kernel that walks downwards
        // keep every prefetched address inside the arrays: a neighbour offset reaches at most one
        // x-layer + one row + one cell beyond the target cell, so stay that far from both ends
        const long long margin = (long long)a.g.ny * a.g.nz + a.g.nz + 1;
        if (!a.pf_strided) {
            const long long t = (long long)i + a.pf;   // 64-bit: N may be close to 2^31
            if (t >= margin && t + margin < a.g.n && t < a.end && t >= a.first) {
                if constexpr (SOA) {
                    const int ti = (int)t;
                    static_for<Q>([&](auto kc) { asm volatile("prefetch.global.L2 [%0];" ::"l"(a.lp[kc] + ti)); });
                } else {
                    const char* q = reinterpret_cast<const char*>(a.src + t * Q);
                    static_for<Q>([&](auto kc) { asm volatile("prefetch.global.L2 [%0];" ::"l"(q + a.ldo[kc])); });
                }
            }
        } else if constexpr (SOA) {
            constexpr int CPL = 128 / sizeof(T);   // cells per line
            const int lane = threadIdx.x & 31;
            const long long tgt = (long long)(i - lane) + a.pf + (long long)lane * CPL;
            if ((((i - a.first) >> 5) % CPL) == 0 && tgt >= margin && tgt + CPL + margin < a.g.n && tgt + CPL < a.end && tgt >= a.first) {
                const int ti = (int)tgt;
                static_for<Q>([&](auto kc) { asm volatile("prefetch.global.L2 [%0];" ::"l"(a.lp[kc] + ti)); });
            }
        }
    }
    T f[Q];
    load_cell<T, Q, SOA, LOAD>(a, i, cs.masked, cs.mask, f);
    collide<Q, MODEL, SHIFT>(f, a.rt);
    store_cell<T, Q, SOA, STORE>(a, i, cs.masked, cs.mask, f);
}

// thread -> cell of the AoS neighbour kernels: a block of 32 * PY threads covers PY z-row segments of 32
// cells with consecutive y (grid: ceil(nz/32) x ceil(ny/PY) x nx), see step_kernel_aos_pull_patch.  Returns
// the cell index, or g.n ("no cell": cell_state makes the lane inactive) outside the box.
#ifndef LBM_AOS_PATCH_PY
#define LBM_AOS_PATCH_PY 4
#endif
template <int PY>
__device__ __forceinline__ int patch_cell(const Geo& g)
{
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int z = blockIdx.x * 32 + lane, y = blockIdx.y * PY + w, x = blockIdx.z;
    if (z >= g.nz || y >= g.ny) return g.n;
    return (x * g.ny + y) * g.nz + z;
}
inline dim3 patch_grid(const Geo& g, int py) { return dim3((g.nz + 31) / 32, (g.ny + py - 1) / py, g.nx); }

// AoS, neighbour side.  A warp that pulls "slot k of 32 consecutive cells" touches 32 different 32-byte
// sectors and uses 4 or 8 bytes of each; ncu (profiles/r02_aos_*) shows the AoS gathers running at the
// rate the LSU / L2 deliver such sectors, not at the DRAM rate.  The internal slot order of a record
// (Lat<Q>::aos_slot) puts the three directions that share (cx, cy) next to each other, so the values a
// warp of bulk cells pulls from ONE neighbouring z-row are the adjacent triples (cz = -1, 0, +1) of 32
// consecutive records: lane l needs slot 1 + s*dz of record l - dz (s = +1 pull, -1 AA pull).  The
// warp therefore loads those 96 values with three requests in which consecutive lanes read consecutive
// addresses (lane -> (record e/3, slot e%3), e = 32j + lane: 11-14 sectors per request instead of
// 32, every byte used), parks them in 96 elements of shared memory and each lane picks its three; only
// the two values that come from the records beyond the ends of the run (lane 0: record -1, lane 31:
// record 32) are fetched directly.  Directions alone in their (cx, cy) group (D3Q19: cz = 0 diagonals)
// are loaded per thread as before.  Every lane of the warp must call this (bulk warps only).
template <class T, int Q, int LOAD>
__device__ __forceinline__ void load_cell_aos_coop(const StepArgs<T>& a, int i, T* __restrict__ scratch, T (&f)[Q])
{
    static_assert(LOAD == LD_PULL || LOAD == LD_AAPULL, "neighbour loads only");
    using L = Lat<Q>;
    const int lane = threadIdx.x & 31;
    const T* __restrict__ src = a.src;
    const long long b = (long long)i - lane;   // first cell of the warp
    const long long A = (long long)a.g.ny * a.g.nz;
    static_for<9>([&](auto gc) {
        constexpr int gx = gc / 3 - 1, gy = gc % 3 - 1;
        // directions of this (cx, cy) group, by cz
        constexpr int km = L::dir_of_code((gx + 1) * 9 + (gy + 1) * 3 + 0);
        constexpr int k0 = L::dir_of_code((gx + 1) * 9 + (gy + 1) * 3 + 1);
        constexpr int kp = L::dir_of_code((gx + 1) * 9 + (gy + 1) * 3 + 2);
        const long long R0 = b - (gx * A + gy * (long long)a.g.nz);   // record that lane 0 pulls its cz = 0 value from
        if constexpr (km >= 0 && kp >= 0) {
            // the triple lives in the group (gx, gy) of the source record (pull) or in (-gx, -gy) (AA pull: slot kbar)
            constexpr int gs = LOAD == LD_PULL ? L::aos_slot(km) : L::aos_slot(L::opp(kp));
            static_for<3>([&](auto jc) {
                const int e = 32 * jc + lane, rec = e / 3, sl = e - 3 * rec;
                scratch[e] = src[(R0 + rec) * Q + gs + sl];
            });
            __syncwarp();
            static_for<3>([&](auto dc) {
                constexpr int dz = dc - 1;
                constexpr int k = dz < 0 ? km : dz == 0 ? k0 : kp;
                constexpr int t = LOAD == LD_PULL ? 1 + dz : 1 - dz;
                const int r = lane - dz;
                T v;
                if (r >= 0 && r < 32) v = scratch[3 * r + t];
                else v = src[(R0 + r) * Q + gs + t];
                f[k] = v;
            });
            __syncwarp();
        } else if constexpr (k0 >= 0) {
            constexpr int sl = LOAD == LD_PULL ? L::aos_slot(k0) : L::aos_slot(L::opp(k0));
            f[k0] = src[(R0 + lane) * Q + sl];
        }
    });
}

// The same for the scatter of the AA odd step (ST_PUSH: pop_k(x + c_k) <- f_out_k): lane l writes slot
// 1 + dz of record l + dz of the destination z-row.  The lanes park their triples in shared memory and the
// warp stores the 96 values with three requests of consecutive addresses; the two entries whose source
// lies in the neighbouring warps (record 0 slot 2, record 31 slot 0) are skipped -- those warps write
// them, as this one writes the two values that leave its run (lane 0: record -1, lane 31: record 32).
// Every location is still written exactly once.  Bulk warps only, every lane must call.
template <class T, int Q>
__device__ __forceinline__ void store_cell_aos_coop(const StepArgs<T>& a, int i, T* __restrict__ scratch, const T (&f)[Q])
{
    using L = Lat<Q>;
    const int lane = threadIdx.x & 31;
    T* __restrict__ dst = a.dst;
    const long long b = (long long)i - lane;
    const long long A = (long long)a.g.ny * a.g.nz;
    static_for<9>([&](auto gc) {
        constexpr int gx = gc / 3 - 1, gy = gc % 3 - 1;
        constexpr int km = L::dir_of_code((gx + 1) * 9 + (gy + 1) * 3 + 0);
        constexpr int k0 = L::dir_of_code((gx + 1) * 9 + (gy + 1) * 3 + 1);
        constexpr int kp = L::dir_of_code((gx + 1) * 9 + (gy + 1) * 3 + 2);
        const long long D0 = b + (gx * A + gy * (long long)a.g.nz);   // record lane 0 pushes its cz = 0 value into
        if constexpr (km >= 0 && kp >= 0) {
            constexpr int gs = L::aos_slot(km);
            static_for<3>([&](auto dc) {
                constexpr int dz = dc - 1;
                constexpr int k = dz < 0 ? km : dz == 0 ? k0 : kp;
                const int r = lane + dz;
                if (r >= 0 && r < 32) scratch[3 * r + 1 + dz] = f[k];
                else dst[(D0 + r) * Q + gs + 1 + dz] = f[k];
            });
            __syncwarp();
            static_for<3>([&](auto jc) {
                const int e = 32 * jc + lane, rec = e / 3, sl = e - 3 * rec;
                if (e != 2 && e != 93) dst[(D0 + rec) * Q + gs + sl] = scratch[e];
            });
            __syncwarp();
        } else if constexpr (k0 >= 0) {
            constexpr int sl = L::aos_slot(k0);
            dst[(D0 + lane) * Q + sl] = f[k0];
        }
    });
}

// AA odd step in AoS (LD_AAPULL -> ST_PUSH): both sides are neighbour accesses.  Bulk warps gather and
// scatter cooperatively (above), the others per thread.  Launch with blockDim/32 * 96 * sizeof(T) bytes of
// dynamic shared memory.
// register caps as for step_kernel in fp64 (72 / 96 registers); fp32 64 / 85
template <class T, int Q>
constexpr int aos_odd_min_blocks() { return sizeof(T) == 8 ? (Q == 19 ? 7 : 5) : (Q == 19 ? 8 : 6); }
template <class T, int Q, int MODEL, bool PATCH = false>
__global__ void __launch_bounds__(128, (aos_odd_min_blocks<T, Q>())) step_kernel_aos_odd(const StepArgs<T> a)
{
    constexpr bool SHIFT = sizeof(T) == 4;
    extern __shared__ __align__(16) unsigned char scratch_raw[];
    T* scratch = reinterpret_cast<T*>(scratch_raw) + (threadIdx.x >> 5) * 96;
    // PATCH: blocks cover patches of z-rows (patch_cell), so that the source rows of the gather are shared in L1;
    // in place, every location is read and written by exactly one cell (R4), so any thread -> cell map is valid
    const int i = PATCH ? patch_cell<LBM_AOS_PATCH_PY>(a.g) : (int)(blockIdx.x * blockDim.x + threadIdx.x);
    const CellState cs = cell_state(a, i, a.g.n);
    const bool coop = __all_sync(0xffffffffu, cs.active && !cs.masked);
    T f[Q];
    if (coop) {
        load_cell_aos_coop<T, Q, LD_AAPULL>(a, i, scratch, f);
        collide<Q, MODEL, SHIFT>(f, a.rt);
        store_cell_aos_coop<T, Q>(a, i, scratch, f);
    } else if (cs.active) {
        load_cell<T, Q, false, LD_AAPULL>(a, i, cs.masked, cs.mask, f);
        collide<Q, MODEL, SHIFT>(f, a.rt);
        store_cell<T, Q, false, ST_PUSH>(a, i, cs.masked, cs.mask, f);
    }
}

// AoS with shared-memory staging.  In the AoS layout pop[N][Q] the Q values of
// the cells of one block are one contiguous run of blockDim*Q elements, but a warp that reads
// "slot k of 32 consecutive cells" touches 32 different sectors.  Whatever is LOCAL to the cell
// (the loads of 2-pop push / AA even / swap pass 1 / collide-only, the stores of 2-pop pull /
// AA even / swap pass 1 / collide-only) therefore goes through a transposing tile: the run is copied
// between global and shared memory by ONE 1-D TMA bulk copy each way (cp.async.bulk: no registers,
// no per-thread address arithmetic, the whole run in flight at once; ncu showed the earlier
// per-thread copy loop at half the bandwidth of the SoA kernels with 4 loads in flight per thread),
// and each thread works on its own record tile[tid*Q .. tid*Q+Q) (Q is odd, so both 4-byte and
// 8-byte records are free of bank conflicts).  Neighbour accesses (LD_PULL, LD_AAPULL, ST_PUSH) stay
// per-thread gathers / scatters.  A run whose size is not a multiple of 16 bytes (the last block of
// a ragged lattice) is copied by the threads.  Launch with (blockDim*Q + blockDim/32*96)*sizeof(T)
// bytes of dynamic shared memory (the tile and the warps' gather scratch).
__device__ __forceinline__ unsigned aos_smem_addr(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
template <class T, int Q, int MODEL, int LOAD, int STORE>
__global__ void __launch_bounds__(128) step_kernel_aos(const StepArgs<T> a)
{
    static_assert(LOAD == LD_LOCAL || STORE != ST_PUSH, "nothing to stage");
    constexpr bool SHIFT = sizeof(T) == 4;
    using L = Lat<Q>;
    extern __shared__ __align__(128) unsigned char tile_raw[];
    __shared__ __align__(8) unsigned long long bar;
    T* tile = reinterpret_cast<T*>(tile_raw);
    const long long base = (long long)blockIdx.x * blockDim.x;   // first cell of the block
    const int i = (int)base + threadIdx.x;
    const int nb = min((long long)blockDim.x, (long long)a.g.n - base) * Q;   // elements of the block's run
    const unsigned bytes = (unsigned)nb * (unsigned)sizeof(T);
    const bool bulk = (bytes & 15u) == 0u;   // base * Q * sizeof(T) is a multiple of 16 for blocks of 128 cells
    if constexpr (LOAD == LD_LOCAL) {
        if (bulk && threadIdx.x == 0) {
            const unsigned b = aos_smem_addr(&bar);
            asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(b) : "memory");
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
            asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(b), "r"(bytes) : "memory");
            asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                         ::"r"(aos_smem_addr(tile)), "l"(a.src + base * Q), "r"(bytes), "r"(b) : "memory");
        }
    }
    const CellState cs = cell_state(a, i, a.g.n);
    T* rec = tile + threadIdx.x * Q;
    T f[Q];
    if constexpr (LOAD == LD_LOCAL) {
        if (bulk) {
            __syncthreads();   // the barrier is initialised
            const unsigned b = aos_smem_addr(&bar);
            unsigned ok;
            do {
                asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], 0; selp.u32 %0, 1, 0, p; }"
                             : "=r"(ok) : "r"(b) : "memory");
            } while (!ok);
        } else {
            const T* __restrict__ run = a.src + base * Q;
            for (int e = threadIdx.x; e < nb; e += blockDim.x) tile[e] = run[e];
            __syncthreads();
        }
        if (cs.active) static_for<Q>([&](auto kc) { constexpr int sl = L::aos_slot(kc); f[kc] = rec[sl]; });
    } else {
        // bulk warps gather cooperatively (load_cell_aos_coop), the others per thread
        const bool coop = __all_sync(0xffffffffu, cs.active && !cs.masked);
        if (coop) {
            T* scratch = tile + (size_t)blockDim.x * Q + (threadIdx.x >> 5) * 96;
            load_cell_aos_coop<T, Q, LOAD>(a, i, scratch, f);
        } else if (cs.active) {
            load_cell<T, Q, false, LOAD>(a, i, cs.masked, cs.mask, f);
        }
        // the other array is written: solid cells of the run get zeros (never read)
        if (!cs.active) static_for<Q>([&](auto kc) { rec[kc] = T(0); });
    }
    if (cs.active) collide<Q, MODEL, SHIFT>(f, a.rt);
    if constexpr (STORE == ST_PUSH) {
        if (cs.active) store_cell<T, Q, false, STORE>(a, i, cs.masked, cs.mask, f);
    } else {
        if (cs.active) static_for<Q>([&](auto kc) { constexpr int sl = L::aos_slot(STORE == ST_SWAPPED ? L::opp(kc) : (int)kc); rec[sl] = f[kc]; });
        if (bulk) {
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // the records, written by the threads, are read by the TMA unit
            __syncthreads();
            if (threadIdx.x == 0) {
                asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;"
                             ::"l"(a.dst + base * Q), "r"(aos_smem_addr(tile)), "r"(bytes) : "memory");
                asm volatile("cp.async.bulk.commit_group;" ::: "memory");
                asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");   // the tile must outlive the copy
            }
        } else {
            __syncthreads();
            T* __restrict__ run = a.dst + base * Q;
            for (int e = threadIdx.x; e < nb; e += blockDim.x) run[e] = tile[e];
        }
    }
}

// Two-population pull in AoS with a block that covers a PATCH of PY z-row segments (32 cells each) with
// consecutive y instead of 32 * PY consecutive cells.  The values a destination row (x, y) pulls for the
// group (gx, gy) come from the source row (x - gx, y - gy), whose records carry all nine groups; with
// consecutive cells per block every source row is fetched from L2 by up to nine different blocks on
// different SMs, each using a third of a sector or less (ncu: L2 -> L1 sectors >= L1 sectors, i.e. no L1
// hit at all, and the kernel runs at the L2's sector rate).  In a patch the rows y .. y+PY-1 of one block
// want the source rows y-1 .. y+PY of each of the three x-layers, PY + 2 fetches for PY rows instead of
// 3 PY, and the warps of a block issue their loads within the same few hundred cycles, so the repeats hit
// in L1 (or merge with the miss in flight).  Everything else as in step_kernel_aos: cooperative gather of
// the slot triples for bulk warps, masked per-thread path otherwise, results through the transposing
// tile, one bulk store per warp (32 records are contiguous).  Launch with grid (ceil(nz/32), ceil(ny/PY),
// nx), 32 * PY threads and (32 PY Q + 96 PY) * sizeof(T) bytes of dynamic shared memory.
template <class T, int Q, int MODEL, int PY>
__global__ void __launch_bounds__(32 * PY) step_kernel_aos_pull_patch(const StepArgs<T> a)
{
    constexpr bool SHIFT = sizeof(T) == 4;
    using L = Lat<Q>;
    extern __shared__ __align__(128) unsigned char tile_raw[];
    T* tile = reinterpret_cast<T*>(tile_raw);
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int z = blockIdx.x * 32 + lane, y = blockIdx.y * PY + w, x = blockIdx.z;
    const bool inside = z < a.g.nz && y < a.g.ny;
    const long long il = ((long long)x * a.g.ny + y) * a.g.nz + z;
    const int i = inside ? (int)il : a.g.n;      // a.g.n: "no cell" for cell_state
    const CellState cs = cell_state(a, i, a.g.n);
    T* rec = tile + threadIdx.x * Q;
    T f[Q];
    const bool coop = __all_sync(0xffffffffu, cs.active && !cs.masked);
    if (coop) {
        T* scratch = tile + (size_t)(32 * PY) * Q + w * 96;
        load_cell_aos_coop<T, Q, LD_PULL>(a, i, scratch, f);
    } else if (cs.active) {
        load_cell<T, Q, false, LD_PULL>(a, i, cs.masked, cs.mask, f);
    }
    if (cs.active) {
        collide<Q, MODEL, SHIFT>(f, a.rt);
        static_for<Q>([&](auto kc) { constexpr int sl = L::aos_slot(kc); rec[sl] = f[kc]; });
    } else {
        static_for<Q>([&](auto kc) { rec[kc] = T(0); });   // solid cells of the written array: zeros (never read)
    }
    // the warp's 32 records are one contiguous run of the other array
    const long long first = il - lane;           // first cell of the warp's run
    const bool whole = blockIdx.x * 32 + 32 <= a.g.nz && y < a.g.ny;     // warp-uniform
    const bool bulk = whole && ((first * Q * (long long)sizeof(T)) & 15LL) == 0LL;
    if (bulk) {
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // the records are read by the TMA unit
        __syncwarp();
        if (lane == 0) {
            asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;"
                         ::"l"(a.dst + first * Q), "r"(aos_smem_addr(tile + (size_t)w * 32 * Q)), "r"((unsigned)(32 * Q * sizeof(T))) : "memory");
            asm volatile("cp.async.bulk.commit_group;" ::: "memory");
            asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");   // the tile must outlive the copy
        }
    } else if (y < a.g.ny) {
        __syncwarp();
        const int cells = min(32, a.g.nz - blockIdx.x * 32);             // cells of this warp inside the row
        const T* __restrict__ from = tile + (size_t)w * 32 * Q;
        T* __restrict__ run = a.dst + first * Q;
        for (int e = lane; e < cells * Q; e += 32) run[e] = from[e];
    }
}

// ------------------------------------------------------------------ swap scheme, pass 2
// After pass 1 pop_kbar(x) holds f_out_k(x).  For the half set k < NH (R5): exchange pop_kbar(x)
// with pop_k(x + c_k) when that neighbour is fluid, else add w_k in place (the value already sits
// in the slot Eq 3 sends it to); and when the neighbour at x - c_k is a wall, add w_kbar to pop_k(x).
// Every slot is touched by exactly one thread (Table 1), so all loads
// are issued before the first store.
// resident blocks of 256 threads per SM for pass 2 (register cap), tuned on B200: fp64 3 / 2 (D3Q19 / D3Q27),
// fp32 4 / 3; the D3Q27 fp64 instance 128 x 5 (96 registers).  Uncapped it took 144 registers (one block of 256
// per SM, 65 % of the copy rate).
#ifndef LBM_SWAP_MAXT_D27
#define LBM_SWAP_MAXT_D27 128
#endif
#ifndef LBM_SWAP_MINB_D27
#define LBM_SWAP_MINB_D27 5
#endif
template <class T, int Q>
constexpr int swap_max_threads() { return (sizeof(T) == 8 && Q == 27) ? LBM_SWAP_MAXT_D27 : 256; }
template <class T, int Q>
constexpr int swap_min_blocks() { return (sizeof(T) == 8 && Q == 27) ? LBM_SWAP_MINB_D27 : (sizeof(T) == 8 ? 3 : 4) - (Q == 27 ? 1 : 0); }
// The half set is dealt over G thread groups (blockIdx.y): a thread then moves only every G-th pair
// of one cell, needs few registers and the SM holds many more of them, at the price of reading
// the cell's code byte G times.  Measured on B200 (256^3 D3Q19 / 192^3 D3Q27, whole swap step, of
// the copy rate): fp64 G = 1: 93.8 / 86.0 %, G = 2: 95.8 / 89.3 %, G = 3: 89.1 / 89.5 %, G = 5:
// 82.1 / 83.4 %; fp32 G = 1: 83.2 / 77.1 %, G = 2: 82.3 / 78.4 %.
#ifndef LBM_SWAP_G_F64
#define LBM_SWAP_G_F64 2
#endif
#ifndef LBM_SWAP_G_F32
#define LBM_SWAP_G_F32 1
#endif
template <class T, int Q>
constexpr int swap_groups() { return sizeof(T) == 8 ? LBM_SWAP_G_F64 : (Q == 27 ? 2 : LBM_SWAP_G_F32); }  // fp32 D3Q27: 82.5 -> 86.6 %
template <class T, int Q, bool SOA, int G, int GI>
__device__ __forceinline__ void swap_pairs(const StepArgs<T>& a, int i, const CellState& cs)
{
    using L = Lat<Q>;
    T* __restrict__ pop = a.dst;
    const Geo& g = a.g;
    T va[L::NH], vb[L::NH];
    if (!cs.masked) {
        static_for<L::NH>([&](auto kc) {
            constexpr int k = kc, kb = L::opp(k);
            if constexpr (k % G == GI) {
                va[k] = pop[slot<SOA, Q, kb>(g, i)];
                vb[k] = pop[slot<SOA, Q, k>(g, (long long)i + offset<Q, k>(g))];
            }
        });
        static_for<L::NH>([&](auto kc) {
            constexpr int k = kc, kb = L::opp(k);
            if constexpr (k % G == GI) {
                pop[slot<SOA, Q, kb>(g, i)] = vb[k];
                pop[slot<SOA, Q, k>(g, (long long)i + offset<Q, k>(g))] = va[k];
            }
        });
    } else {
        // a link to a solid neighbour exchanges nothing: slot kbar of this cell keeps its value
        // (plus w_k), and slot k of this cell is read and rewritten with w_kbar added when the
        // neighbour at x - c_k is a moving wall
        const Edge e(cs.mask, g);
        static_for<L::NH>([&](auto kc) {
            constexpr int k = kc, kb = L::opp(k);
            if constexpr (k % G == GI) {
                const bool sol = e.template solid_at<Q, k>();
                const long long pb = sol ? slot<SOA, Q, k>(g, i) : slot<SOA, Q, k>(g, (long long)i + e.template off<Q, k, +1>(g));
                va[k] = pop[slot<SOA, Q, kb>(g, i)];
                vb[k] = pop[pb];
            }
        });
        static_for<L::NH>([&](auto kc) {
            constexpr int k = kc, kb = L::opp(k);
            if constexpr (k % G == GI) {
                const bool sol = e.template solid_at<Q, k>();
                const bool back_moving = e.template moving_at<Q, kb>();   // neighbour at x - c_k
                const long long pa = slot<SOA, Q, kb>(g, i);
                if (!sol) {
                    const long long pb = slot<SOA, Q, k>(g, (long long)i + e.template off<Q, k, +1>(g));
                    pop[pa] = vb[k];
                    pop[pb] = va[k];
                    // pop_k(x) belongs to the exchange of the cell at x - c_k unless that one is solid
                    if (back_moving) pop[slot<SOA, Q, k>(g, i)] += a.wterm[kb];
                } else {
                    // vb[k] holds pop_k(x) here
                    if (e.template moving_at<Q, k>()) pop[pa] = va[k] + a.wterm[k];
                    if (back_moving) pop[slot<SOA, Q, k>(g, i)] = vb[k] + a.wterm[kb];
                }
            }
        });
    }
}

// Swap pass 2 in AoS for a warp of bulk cells: the pairs of one (cx, cy) group of the half set are the
// adjacent slot triples of 32 consecutive records on BOTH sides (own records: slots of kbar; the
// neighbouring z-row: slots of k, shifted by cz), so they move with requests of consecutive addresses
// through 2 x 96 elements of shared memory (see load_cell_aos_coop / store_cell_aos_coop); the pairs
// alone in their group are exchanged per thread.  All loads of a group precede its stores, and no two
// groups touch the same slot.  Every lane must call.
template <class T, int Q>
__device__ __forceinline__ void swap_pairs_aos_coop(const StepArgs<T>& a, int i, T* __restrict__ sa, T* __restrict__ sb)
{
    using L = Lat<Q>;
    const int lane = threadIdx.x & 31;
    T* __restrict__ pop = a.dst;
    const long long b = (long long)i - lane;
    const long long A = (long long)a.g.ny * a.g.nz;
    static_for<9>([&](auto gc) {
        constexpr int gx = gc / 3 - 1, gy = gc % 3 - 1;
        constexpr int km = L::dir_of_code((gx + 1) * 9 + (gy + 1) * 3 + 0);
        constexpr int k0 = L::dir_of_code((gx + 1) * 9 + (gy + 1) * 3 + 1);
        constexpr int kp = L::dir_of_code((gx + 1) * 9 + (gy + 1) * 3 + 2);
        const long long D0 = b + (gx * A + gy * (long long)a.g.nz);
        // a whole group belongs to the half set or to its opposite, except (0, 0, .), where only cz = -1 does
        if constexpr (km >= 0 && kp >= 0 && k0 >= 0 && km < L::NH && k0 < L::NH && kp < L::NH) {
            constexpr int gs = L::aos_slot(km);            // neighbour side: slots of k = (gx, gy, dz): gs + 1 + dz
            constexpr int go = L::aos_slot(L::opp(kp));    // own side: slots of kbar = (-gx, -gy, -dz): go + 1 - dz
            static_for<3>([&](auto jc) {
                const int e = 32 * jc + lane, rec = e / 3, sl = e - 3 * rec;
                sa[e] = pop[(b + rec) * Q + go + sl];
                sb[e] = pop[(D0 + rec) * Q + gs + sl];
            });
            __syncwarp();
            T va[3], vb[3];
            static_for<3>([&](auto dc) {
                constexpr int dz = dc - 1;
                const int r = lane + dz;
                va[dc] = sa[3 * lane + 1 - dz];
                vb[dc] = (r >= 0 && r < 32) ? sb[3 * r + 1 + dz] : pop[(D0 + r) * Q + gs + 1 + dz];
            });
            __syncwarp();
            static_for<3>([&](auto dc) {
                constexpr int dz = dc - 1;
                const int r = lane + dz;
                sa[3 * lane + 1 - dz] = vb[dc];
                if (r >= 0 && r < 32) sb[3 * r + 1 + dz] = va[dc];
                else pop[(D0 + r) * Q + gs + 1 + dz] = va[dc];
            });
            __syncwarp();
            static_for<3>([&](auto jc) {
                const int e = 32 * jc + lane, rec = e / 3, sl = e - 3 * rec;
                pop[(b + rec) * Q + go + sl] = sa[e];
                if (e != 2 && e != 93) pop[(D0 + rec) * Q + gs + sl] = sb[e];
            });
            __syncwarp();
        } else {
            static_for<3>([&](auto dc) {
                constexpr int dz = dc - 1;
                constexpr int k = dz < 0 ? km : dz == 0 ? k0 : kp;
                if constexpr (k >= 0 && k < L::NH) {
                    constexpr int kb = L::opp(k);
                    const long long pa = ((long long)i) * Q + L::aos_slot(kb);
                    const long long pb = ((long long)i + offset<Q, k>(a.g)) * Q + L::aos_slot(k);
                    const T x = pop[pa], y = pop[pb];
                    pop[pa] = y;
                    pop[pb] = x;
                }
            });
        }
    });
}

// swap pass 2, AoS: bulk warps exchange cooperatively, the others per thread (one thread group).  Launch
// with blockDim/32 * 192 * sizeof(T) bytes of dynamic shared memory.
// (blocks over patches of z-rows as in step_kernel_aos_odd were measured here too: no gain, 256^3 D3Q19 fp64
// 3.557 -> 3.568 ms, D3Q27 cumulants 2.09 -> 2.30 ms; pass 2 keeps consecutive cells per block)
template <class T, int Q>
__global__ void __launch_bounds__(128) swap_stream_kernel_aos(const StepArgs<T> a)
{
    extern __shared__ __align__(16) unsigned char swap_scratch_raw[];
    T* sa = reinterpret_cast<T*>(swap_scratch_raw) + (threadIdx.x >> 5) * 192;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const CellState cs = cell_state(a, i, a.g.n);
    const bool coop = __all_sync(0xffffffffu, cs.active && !cs.masked);
    if (coop) swap_pairs_aos_coop<T, Q>(a, i, sa, sa + 96);
    else if (cs.active) swap_pairs<T, Q, false, 1, 0>(a, i, cs);
}

template <class T, int Q, bool SOA, int G>
// (two groups, D3Q27: 4 / 5 blocks of 256 = 64 / 48 registers; at 5 / 6 the fp64 instance spilled 136 bytes.
// Same box, 192^3 D3Q27 swap fp64: BGK-W2 95.2 -> 97.6 %, cumulants 94.8 -> 97.0 %; fp32 86.9 -> 87.2 %)
__global__ void __launch_bounds__(G == 1 ? swap_max_threads<T, Q>() : 256, G == 1 ? swap_min_blocks<T, Q>() : (sizeof(T) == 8 ? (Q == 27 ? 4 : 5) : (Q == 27 ? 5 : 6)))
swap_stream_kernel(const StepArgs<T> a)
{
    asm volatile("griddepcontrol.launch_dependents;");   // see step_kernel
    const unsigned blk = a.rev ? gridDim.x - 1u - blockIdx.x : blockIdx.x;   // see step_kernel
    const int i = blk * blockDim.x + threadIdx.x;
    const CellState cs = cell_state<false>(a, i, a.g.n);
    asm volatile("griddepcontrol.wait;" ::: "memory");
    if (!cs.active) return;
    static_for<G>([&](auto gc) {
        if (blockIdx.y == (unsigned)gc) {
            // L2 prefetch, see step_kernel (offsets of the half set point forward only): per thread in fp64,
            // one warp in 32 with a line per lane in fp32 (pass 2 in fp32 ran at 77 % of the copy rate with
            // 18 prefetch instructions in every thread)
            const long long reach = (long long)a.g.ny * a.g.nz + a.g.nz + 1;
            if constexpr (sizeof(T) == 8) {
                if (a.pf != 0 && (long long)i + a.pf >= 0 && (long long)i + a.pf + reach < a.g.n) {   // pf < 0: walking downwards
                    using L = Lat<Q>;
                    static_for<L::NH>([&](auto kc) {
                        constexpr int k = kc, kb = L::opp(k);
                        if constexpr (k % G == gc) {
                            asm volatile("prefetch.global.L2 [%0];" ::"l"(a.dst + slot<SOA, Q, kb>(a.g, (long long)i + a.pf)));
                            asm volatile("prefetch.global.L2 [%0];" ::"l"(a.dst + slot<SOA, Q, k>(a.g, (long long)i + a.pf + offset<Q, k>(a.g))));
                        }
                    });
                }
            } else if (a.pf != 0) {
                constexpr int CPL = 128 / sizeof(T);   // cells per line
                const int lane = threadIdx.x & 31;
                const long long tgt = (long long)(i - lane) + a.pf + (long long)lane * CPL;
                if (((i >> 5) % CPL) == 0 && tgt >= 0 && tgt + CPL + reach < a.g.n) {
                    using L = Lat<Q>;
                    static_for<L::NH>([&](auto kc) {
                        constexpr int k = kc, kb = L::opp(k);
                        if constexpr (k % G == gc) {
                            asm volatile("prefetch.global.L2 [%0];" ::"l"(a.dst + slot<SOA, Q, kb>(a.g, tgt)));
                            asm volatile("prefetch.global.L2 [%0];" ::"l"(a.dst + slot<SOA, Q, k>(a.g, tgt + offset<Q, k>(a.g))));
                        }
                    });
                }
            }
            swap_pairs<T, Q, SOA, G, gc>(a, i, cs);
        }
    });
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
    static_for<Q>([&](auto kc) { pop[slot<SOA, Q, kc>(g, i)] = E[kc]; });
}

// rho, u of the pre-collision state; LOAD says where that state lives
template <class T, int Q, bool SOA, int LOAD>
__global__ void macroscopic_kernel(const T* __restrict__ pop, const uint8_t* __restrict__ code, Geo g,
                                   StepArgs<T> a, T* __restrict__ rho, T* __restrict__ u)
{
    constexpr bool SHIFT = sizeof(T) == 4;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const CellState cs = cell_state(a, i, g.n);
    if (i >= g.n) return;
    T r = T(0), uu[3] = {T(0), T(0), T(0)};
    if (cs.active) {
        T f[Q], dr;
        load_cell<T, Q, SOA, LOAD>(a, i, cs.masked, cs.mask, f);
        moments_rho_u<Q, SHIFT>(f, r, dr, uu);
    }
    rho[i] = r;
    u[i] = uu[0];
    u[(long long)g.n + i] = uu[1];
    u[2LL * g.n + i] = uu[2];
}

// kinetic energy, stage 1: one cell per thread, one double per block of 256 cells (fixed tree: warp
// shuffle, then warp 0), so that as many loads are in flight as in the step kernels
template <class T, int Q, bool SOA, int LOAD>
__global__ void __launch_bounds__(256, sizeof(T) == 8 ? (Q == 19 ? 3 : 2) : (Q == 19 ? 6 : 4)) energy_kernel(const T* __restrict__ pop, const uint8_t* __restrict__ code, Geo g,
                                                                         StepArgs<T> a, double* __restrict__ partial)
{
    constexpr bool SHIFT = sizeof(T) == 4;
    double e = 0.0;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const CellState cs = cell_state(a, i, g.n);
    if (cs.active) {
        T f[Q], r, dr, uu[3];
        load_cell<T, Q, SOA, LOAD>(a, i, cs.masked, cs.mask, f);
        moments_rho_u<Q, SHIFT>(f, r, dr, uu);
        e = 0.5 * (double)r * ((double)uu[0] * uu[0] + (double)uu[1] * uu[1] + (double)uu[2] * uu[2]);
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
// cells == nullptr: the whole plane (out[i], i < n); else a gather of m listed cells (out[t] = f_k(cells[t]))
template <class T, int Q, bool SOA>
__global__ void extract_plane_kernel(const T* __restrict__ pop, const uint8_t* __restrict__ code, Geo g, PlaneArgs p,
                                     T* __restrict__ out, const int* __restrict__ cells, int m)
{
    constexpr bool SHIFT = sizeof(T) == 4;
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= m) return;
    const int i = cells ? cells[t] : t;
    T v = T(0);
    if (!(code[i] & 3)) {
        int n = i;
        if (p.sx | p.sy | p.sz) {
            const int z = i % g.nz, y = (i / g.nz) % g.ny, x = i / (g.nz * g.ny);
            n = (wrap1(x - p.sx, g.nx) * g.ny + wrap1(y - p.sy, g.ny)) * g.nz + wrap1(z - p.sz, g.nz);
        }
        const int nc = code[n] & 3;
        if (nc == 0 || nc == CODE_GHOST) v = pop[slot_raw<SOA, Q>(g, p.slot_fluid, n)];
        else v = pop[slot_raw<SOA, Q>(g, p.slot_wall, i)] + (nc == CODE_MOVING ? T(p.wterm) : T(0));
        if (SHIFT) v += T(p.weight);
    }
    out[t] = v;
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
    pop[slot_raw<SOA, Q>(g, k, i)] = v;
}

// halo exchange of the slab decomposition along x: one x-layer (ny*nz contiguous
// cells in SoA) of `ndir` population planes to (PACK) or from a contiguous buffer [ndir][ny*nz].
// Raw stored values (fp32: shifted), so both ends must have the same dtype.
//
//   slot[d]     population plane of the d-th direction of the message (k, or kbar where the scheme
//               keeps post-collision values in the opposite slot: AA even, swap pass 1)
//   first       index of the first cell of the layer read (PACK) or written (unpack)
//   merge != 0  (unpack only) the message holds values that a neighbouring slab would have pushed or
//               exchanged into this slab's outermost OWNED layer (AA odd step, swap pass 2): cell x
//               of that layer takes direction d only when its upstream cell x - c_d, which lies in
//               the ghost layer starting at `up_first`, is a GHOST cell (fluid on the neighbour); a
//               solid upstream cell means x has bounced that population back itself.
//               merge == 1: the buffer is indexed by the destination cell, == 2: by the upstream cell.
//   flag        PACK: when not null the buffer is the RECEIVE buffer of the neighbouring slab (peer
//               memory, written over NVLink), and the block that finishes last publishes `seq`
//               there with system scope; unpack: when not null, wait until *flag >= seq first.
struct HaloArgs {
    int slot[9];
    int cy[9], cz[9];
    int ndir;
    long long first, up_first;
    int ny, nz;
    int cells;         // ny*nz
    int merge;
    unsigned long long* flag;
    unsigned long long seq;
    unsigned* counter;   // PACK + flag: blocks done so far (sender's memory, zero between launches)
    int* status;         // unpack + flag: set to 1 when the wait gave up
};
__device__ __forceinline__ unsigned long long ld_acquire_sys(const unsigned long long* p)
{
    unsigned long long v;
    asm volatile("ld.acquire.sys.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
template <class T, bool PACK>
__global__ void __launch_bounds__(256) halo_kernel(T* __restrict__ pop, const uint8_t* __restrict__ code, long long stride,
                                                   HaloArgs p, T* __restrict__ buf)
{
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    const int d = blockIdx.y;
    if (!PACK && p.flag) {   // the message must have landed (bounded wait: a lost neighbour must not hang the GPU)
        __shared__ int ok;
        if (threadIdx.x == 0) {
            int good = 0;
            for (long long spin = 0; spin < (1LL << 24); ++spin) {
                if (ld_acquire_sys(p.flag) >= p.seq) { good = 1; break; }
                __nanosleep(64);
            }
            if (!good) *p.status = 1;
            ok = good;
        }
        __syncthreads();
        if (!ok) return;
    }
    if (t < p.cells) {
        T* b = buf + (long long)d * p.cells + t;
        T* slot = pop + (long long)p.slot[d] * stride + p.first + t;
        if (PACK) {
            *b = *slot;
        } else if (!p.merge) {
            *slot = *b;
        } else {
            const int iy = t / p.nz, iz = t - iy * p.nz;
            const int up = wrap1(iy - p.cy[d], p.ny) * p.nz + wrap1(iz - p.cz[d], p.nz);
            if (code[p.up_first + up] == CODE_GHOST && !(code[p.first + t] & 3))
                *slot = buf[(long long)d * p.cells + (p.merge == 2 ? up : t)];
        }
    }
    if (PACK && p.flag) {   // publish: every block's stores first, then the sequence number
        __threadfence_system();
        __syncthreads();
        if (threadIdx.x == 0) {
            const unsigned total = gridDim.x * gridDim.y;
            if (atomicAdd(p.counter, 1u) == total - 1u) {
                *p.counter = 0u;
                __threadfence_system();
                asm volatile("st.release.sys.global.u64 [%0], %1;" ::"l"(p.flag), "l"(p.seq) : "memory");
            }
        }
    }
}

}  // namespace lbm
