// lattice.cuh -- compile-time D3Q19 / D3Q27 velocity sets for the CUDA path.
//
// Direction order is the canonical ABI order of include/lbm.h (reading R7, anchored on
// PAPER.md:L325 "c_0 = (-1,0,0) = -c_10"): a half set, the rest velocity, then the negatives of
// the half set in the same order, so that opp(k) = k + NH + 1 for k < NH.  Weights are the textbook
// ones (R8; c_s^2 = 1/3).  Everything here is constexpr so that fully unrolled
// kernels see only immediates (the paper's "unrolled" code version).
#pragma once
#include <cstdint>
#include <type_traits>
#include <utility>

namespace lbm {

#define LBM_HD __host__ __device__ __forceinline__

// compile-time integer usable in device code (std::integral_constant's conversion is host-only)
template <int I>
struct IC {
    static constexpr int value = I;
    LBM_HD constexpr operator int() const { return I; }
};

// compile-time loop: f(IC<I>) for I in [0, N)
template <class F, int... I>
LBM_HD constexpr void static_for_impl(F&& f, std::integer_sequence<int, I...>)
{
    (f(IC<I>{}), ...);
}
template <int N, class F>
LBM_HD constexpr void static_for(F&& f)
{
    static_for_impl(static_cast<F&&>(f), std::make_integer_sequence<int, N>{});
}

template <int Q>
struct Lat {
    static_assert(Q == 19 || Q == 27, "D3Q19 or D3Q27");
    static constexpr int NH = (Q - 1) / 2;  // size of the half set
    static constexpr int REST = NH;

    // half-set velocities, packed as (cx+1)*9 + (cy+1)*3 + (cz+1)
    LBM_HD static constexpr int half_code(int h)
    {
        // (-1,0,0) (0,-1,0) (0,0,-1) (-1,-1,0) (-1,1,0) (-1,0,-1) (-1,0,1) (0,-1,-1) (0,-1,1)
        // (-1,-1,-1) (-1,-1,1) (-1,1,-1) (-1,1,1)
        constexpr int codes[13] = {4, 10, 12, 1, 7, 3, 5, 9, 11, 0, 2, 6, 8};
        return codes[h];
    }
    // grid code g = (cx+1)*9 + (cy+1)*3 + (cz+1) of direction k
    LBM_HD static constexpr int code(int k)
    {
        return k < NH ? half_code(k) : k == NH ? 13 : 26 - half_code(k - NH - 1);
    }
    LBM_HD static constexpr int cx(int k) { return code(k) / 9 - 1; }
    LBM_HD static constexpr int cy(int k) { return (code(k) / 3) % 3 - 1; }
    LBM_HD static constexpr int cz(int k) { return code(k) % 3 - 1; }
    LBM_HD static constexpr int opp(int k) { return k < NH ? k + NH + 1 : k == NH ? NH : k - NH - 1; }
    LBM_HD static constexpr int norm2(int k) { return cx(k) * cx(k) + cy(k) * cy(k) + cz(k) * cz(k); }
    // direction index of grid code g, or -1 when the lattice has no such velocity
    LBM_HD static constexpr int dir_of_code(int g)
    {
        for (int k = 0; k < Q; ++k)
            if (code(k) == g) return k;
        return -1;
    }
    // slot of direction k inside an AoS record (internal order, free by R7): directions sorted by their
    // grid code, i.e. by (cx, cy) first and cz last, so that the (up to) three directions that share
    // (cx, cy) sit next to each other in the order cz = -1, 0, +1.  The populations a cell pulls from
    // one neighbouring z-row then form adjacent triples of consecutive records (kernels.cuh, cooperative
    // AoS gather).  D3Q27: the grid code itself.
    LBM_HD static constexpr int aos_slot(int k)
    {
        int r = 0;
        for (int j = 0; j < Q; ++j)
            if (code(j) < code(k)) ++r;
        return r;
    }
    // weight t_k
    LBM_HD static constexpr double w(int k)
    {
        const int n2 = norm2(k);
        if (Q == 19) return n2 == 0 ? 1.0 / 3.0 : n2 == 1 ? 1.0 / 18.0 : 1.0 / 36.0;
        return n2 == 0 ? 8.0 / 27.0 : n2 == 1 ? 2.0 / 27.0 : n2 == 2 ? 1.0 / 54.0 : 1.0 / 216.0;
    }
    // is the moment (p,q,r) in the lattice's moment set (Eq 8 / Eq 12)?
    LBM_HD static constexpr bool has_moment(int p, int q, int r)
    {
        return Q == 27 || p == 0 || q == 0 || r == 0;
    }
};

}  // namespace lbm
