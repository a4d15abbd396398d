// collision.cuh -- the collision operator Omega (Eq 1) of the ten models, written
// matrix-free and fully unrolled (the paper's "unrolled" code version; moments
// to populations "without matrices", Eq 8-10), entirely in registers.
//
//   W2 family   BGK_W2 (Eq 6-7 with the opposite-pair shortcut), TRT (R15),
//               REG (R18): closed forms per opposite pair.
//   moment hub  BGK_NW4, RM, HM, CM, CHM, K, RR (Eq 11-15): populations
//               -> raw moments by three one-dimensional sweeps over the 3x3x3 velocity grid (the
//               tensor-product form of Eq 12), raw -> model basis by per-axis triangular maps
//               (binomial shift for central moments, H_2 = c^2 - c_s^2 for Hermite), relaxation
//               (Eq 11, Eq 13-15), and the same maps backwards.  On D3Q19 only the 19 moments of
//               Eq 8 exist; the 8 raw moments with p,q,r >= 1 are identically zero for a
//               19-velocity population and are kept zero on the way back, which is exactly the
//               inverse that Eq 8-10 write out.
//
// SHIFT = true works on g_k = f_k - t_k (the round-off mitigation the paper points to at
// PAPER.md:L106, reading R20): rho - 1 = sum g_k; raw moments of g are those of f minus the
// rest-state moments prod {1, 0, c_s^2}.
#pragma once
#include "lattice.cuh"
#include "cumulants_gen.cuh"

namespace lbm {

enum Model { M_BGK_W2 = 0, M_BGK_NW4, M_TRT, M_RM, M_HM, M_CM, M_CHM, M_K, M_RR, M_REG,
             // the same five moment-space models compiled for "every moment of order >= 3 relaxed with
             // exactly 1": their post-collision value is the equilibrium, so the
             // pre-collision moments of those orders are never computed
             M_EQHI_FIRST, M_RM_E = M_EQHI_FIRST, M_HM_E, M_CM_E, M_CHM_E, M_K_E, M_COUNT };

__host__ __device__ constexpr bool model_eq_hi(int model) { return model >= M_EQHI_FIRST; }
// the model a variant computes
__host__ __device__ constexpr int model_base(int model) { return model >= M_EQHI_FIRST ? model - M_EQHI_FIRST + M_RM : model; }
// the variant of a model with orders >= 3 equilibrated, or the model itself when it has none
__host__ __device__ constexpr int model_eq_variant(int model)
{
    return (model >= M_RM && model <= M_K) ? model - M_RM + M_EQHI_FIRST : model;
}

template <class T>
struct Rates {
    T omega;        // shear rate (second-order moments; BGK rate; TRT omega+)
    T omega_bulk;   // Eq 13-15
    T omega3;       // moments of order 3
    T omega_hi;     // moments of order >= 4
    T omega_minus;  // TRT omega-
};

__host__ __device__ constexpr bool model_is_w2(int model)
{
    return model == M_BGK_W2 || model == M_TRT || model == M_REG;
}

// ---------------------------------------------------------------- rho, u
// drho = rho - (SHIFT ? 1 : 0)
template <int Q, bool SHIFT, class T>
__device__ __forceinline__ void moments_rho_u(const T (&f)[Q], T& rho, T& drho, T (&u)[3])
{
    using L = Lat<Q>;
    T s = T(0), jx = T(0), jy = T(0), jz = T(0);
    // pairwise: f_k + f_kbar feeds rho, f_kbar - f_k the momentum (c_kbar = -c_k)
    static_for<L::NH>([&](auto kc) {
        constexpr int k = kc, kb = L::opp(k);
        const T sp = f[k] + f[kb];
        const T sm = f[k] - f[kb];
        s += sp;
        if constexpr (L::cx(k) != 0) jx += T(L::cx(k)) * sm;
        if constexpr (L::cy(k) != 0) jy += T(L::cy(k)) * sm;
        if constexpr (L::cz(k) != 0) jz += T(L::cz(k)) * sm;
    });
    s += f[L::REST];
    drho = s;
    rho = SHIFT ? T(1) + s : s;
    const T inv = T(1) / rho;
    u[0] = jx * inv;
    u[1] = jy * inv;
    u[2] = jz * inv;
}

template <int Q, int K, class T>
__device__ __forceinline__ T c_dot(const T (&u)[3])
{
    using L = Lat<Q>;
    T cu = T(0);
    if constexpr (L::cx(K) != 0) cu += T(L::cx(K)) * u[0];
    if constexpr (L::cy(K) != 0) cu += T(L::cy(K)) * u[1];
    if constexpr (L::cz(K) != 0) cu += T(L::cz(K)) * u[2];
    return cu;
}

// ---------------------------------------------------------------- W2 equilibrium, Eq 6-7
// E[k] - (SHIFT ? t_k : 0)
template <int Q, bool SHIFT, class T>
__device__ __forceinline__ void equilibrium_w2(T rho, T drho, const T (&u)[3], T (&E)[Q])
{
    using L = Lat<Q>;
    const T usq15 = T(1.5) * (u[0] * u[0] + u[1] * u[1] + u[2] * u[2]);
    static_for<L::NH>([&](auto kc) {
        constexpr int k = kc, kb = L::opp(k);
        const T tk = T(L::w(k));
        const T cu = c_dot<Q, k>(u);
        const T quad = T(4.5) * cu * cu - usq15;
        const T sym = SHIFT ? tk * (drho + rho * quad) : tk * rho * (T(1) + quad);
        const T asym = T(3) * tk * rho * cu;
        E[k] = sym + asym;
        E[kb] = sym - asym;  // Eq 7: E_kbar = E_k - 6 rho t_k c_k.u
    });
    const T t0 = T(L::w(L::REST));
    E[L::REST] = SHIFT ? t0 * (drho - rho * usq15) : t0 * rho * (T(1) - usq15);
}

// ---------------------------------------------------------------- moment hub
// m[] is indexed p*9 + q*3 + r.  One sweep turns the three values of a line along AXIS,
// (a_-1, a_0, a_+1), into its 1D raw moments (sum, a_+1 - a_-1, a_+1 + a_-1).
template <int AXIS>
__host__ __device__ constexpr int line_index(int line, int j)
{
    // line enumerates the other two indices (o1 major, o2 minor)
    const int o1 = line / 3, o2 = line % 3;
    return AXIS == 0 ? j * 9 + o1 * 3 + o2 : AXIS == 1 ? o1 * 9 + j * 3 + o2 : o1 * 9 + o2 * 3 + j;
}

template <int AXIS, class T>
__device__ __forceinline__ void sweep_fwd(T (&m)[27])
{
    static_for<9>([&](auto lc) {
        constexpr int i0 = line_index<AXIS>(lc, 0), i1 = line_index<AXIS>(lc, 1), i2 = line_index<AXIS>(lc, 2);
        const T am = m[i0], a0 = m[i1], ap = m[i2];
        const T s2 = ap + am;
        m[i0] = s2 + a0;
        m[i1] = ap - am;
        m[i2] = s2;
    });
}
template <int AXIS, class T>
__device__ __forceinline__ void sweep_bwd(T (&m)[27])
{
    static_for<9>([&](auto lc) {
        constexpr int i0 = line_index<AXIS>(lc, 0), i1 = line_index<AXIS>(lc, 1), i2 = line_index<AXIS>(lc, 2);
        const T m0 = m[i0], m1 = m[i1], m2 = m[i2];
        m[i0] = T(0.5) * (m2 - m1);
        m[i1] = m0 - m2;
        m[i2] = T(0.5) * (m2 + m1);
    });
}

template <int Q, class T>
__device__ __forceinline__ void raw_from_pop(const T (&f)[Q], T (&m)[27])
{
    using L = Lat<Q>;
    static_for<27>([&](auto gc) {
        constexpr int k = L::dir_of_code(gc);
        if constexpr (k >= 0) m[gc] = f[k];
        else m[gc] = T(0);
    });
    sweep_fwd<2>(m);
    sweep_fwd<1>(m);
    sweep_fwd<0>(m);
}
template <int Q, class T>
__device__ __forceinline__ void pop_from_raw(T (&m)[27], T (&f)[Q])
{
    using L = Lat<Q>;
    // D3Q19: the raw moments outside the set of Eq 8 are zero (see the header of this file)
    static_for<27>([&](auto ic) {
        constexpr int p = ic / 9, q = (ic / 3) % 3, r = ic % 3;
        if constexpr (!L::has_moment(p, q, r)) m[ic] = T(0);
    });
    sweep_bwd<0>(m);
    sweep_bwd<1>(m);
    sweep_bwd<2>(m);
    static_for<27>([&](auto gc) {
        constexpr int k = L::dir_of_code(gc);
        if constexpr (k >= 0) f[k] = m[gc];
    });
}

// per-axis triangular maps, applied only to moments inside the lattice's set (a lower set, so
// every input needed by an in-set output is in the set too)
enum { TO_CENTRAL, FROM_CENTRAL, TO_HERMITE, FROM_HERMITE };
template <int Q, int AXIS, int KIND, class T>
__device__ __forceinline__ void axis_map(T (&m)[27], T v)
{
    using L = Lat<Q>;
    static_for<9>([&](auto lc) {
        constexpr int i0 = line_index<AXIS>(lc, 0), i1 = line_index<AXIS>(lc, 1), i2 = line_index<AXIS>(lc, 2);
        constexpr bool in1 = L::has_moment(i1 / 9, (i1 / 3) % 3, i1 % 3);
        constexpr bool in2 = L::has_moment(i2 / 9, (i2 / 3) % 3, i2 % 3);
        if constexpr (KIND == TO_CENTRAL) {  // k1 = m1 - v m0; k2 = m2 - 2 v m1 + v^2 m0
            if constexpr (in1) {
                const T m1 = m[i1];
                const T k1 = m1 - v * m[i0];
                m[i1] = k1;
                if constexpr (in2) m[i2] = m[i2] - v * (m1 + k1);
            }
        } else if constexpr (KIND == FROM_CENTRAL) {  // m1 = k1 + v k0; m2 = k2 + 2 v k1 + v^2 k0
            if constexpr (in1) {
                const T k1 = m[i1];
                const T m1 = k1 + v * m[i0];
                m[i1] = m1;
                if constexpr (in2) m[i2] = m[i2] + v * (m1 + k1);
            }
        } else if constexpr (KIND == TO_HERMITE) {  // H_2 = c^2 - c_s^2
            if constexpr (in2) m[i2] = m[i2] - T(1.0 / 3.0) * m[i0];
        } else {
            if constexpr (in2) m[i2] = m[i2] + T(1.0 / 3.0) * m[i0];
        }
    });
}
template <int Q, int KIND, class T>
__device__ __forceinline__ void basis_map(T (&m)[27], const T (&u)[3])
{
    axis_map<Q, 0, KIND>(m, u[0]);
    axis_map<Q, 1, KIND>(m, u[1]);
    axis_map<Q, 2, KIND>(m, u[2]);
}

// one-dimensional equilibrium factors of order p in each basis (per unit density):
//   raw: 1, v, v^2 + c_s^2     Hermite: 1, v, v^2     central: 1, 0, c_s^2     central Hermite: 1, 0, 0
//   cumulants: c_s^2 for the three diagonal second-order ones, zero for everything else of order >= 2
enum { B_RAW, B_HERMITE, B_CENTRAL, B_CENTRAL_HERMITE, B_CUMULANT };
template <int BASIS, int P, class T>
__device__ __forceinline__ T eq_factor(T v)
{
    if constexpr (P == 0) return T(1);
    else if constexpr (P == 1) return (BASIS == B_RAW || BASIS == B_HERMITE) ? v : T(0);
    else return BASIS == B_RAW ? v * v + T(1.0 / 3.0) : BASIS == B_HERMITE ? v * v
              : (BASIS == B_CENTRAL || BASIS == B_CUMULANT) ? T(1.0 / 3.0) : T(0);
}

// Eq 11 on every moment of order >= 2, Eq 13-15 on the three diagonal second-order ones.
// `scale` multiplies the per-unit-density equilibrium (rho for moments of f, 1 for cumulants).
// EQHI: the rates of every order >= 3 are exactly 1, so those moments are SET to their equilibrium
// (PAPER.md:L340-342); nothing reads their pre-collision values any more and the compiler drops the
// part of the forward transform that produced them (the code is fully unrolled, registers only).
template <int Q, int BASIS, bool EQHI = false, class T>
__device__ __forceinline__ void relax_moments(T (&m)[27], T scale, const T (&u)[3], const Rates<T>& rt)
{
    using L = Lat<Q>;
    const T n200 = m[18] - scale * eq_factor<BASIS, 2>(u[0]);
    const T n020 = m[6] - scale * eq_factor<BASIS, 2>(u[1]);
    const T n002 = m[2] - scale * eq_factor<BASIS, 2>(u[2]);
    const T wm = (rt.omega_bulk - rt.omega) * T(1.0 / 3.0);  // omega_- 
    const T wp = wm + rt.omega;                               // omega_+
    static_for<27>([&](auto ic) {
        constexpr int p = ic / 9, q = (ic / 3) % 3, r = ic % 3, order = p + q + r;
        if constexpr (order >= 2 && L::has_moment(p, q, r) && !(order == 2 && (p == 2 || q == 2 || r == 2))) {
            const T meq = (BASIS == B_CUMULANT)
                              ? T(0)
                              : scale * eq_factor<BASIS, p>(u[0]) * eq_factor<BASIS, q>(u[1]) * eq_factor<BASIS, r>(u[2]);
            if constexpr (EQHI && order >= 3) {
                m[ic] = meq;
            } else {
                const T w = order == 2 ? rt.omega : order == 3 ? rt.omega3 : rt.omega_hi;
                m[ic] = m[ic] - w * (m[ic] - meq);
            }
        }
    });
    m[18] = m[18] - wp * n200 - wm * n020 - wm * n002;  // Eq 13
    m[6] = m[6] - wm * n200 - wp * n020 - wm * n002;    // Eq 14
    m[2] = m[2] - wm * n200 - wm * n020 - wp * n002;    // Eq 15
}

// remove / add the rest-state raw moments prod {1,0,c_s^2} (SHIFT bookkeeping)
template <int Q, int SIGN, class T>
__device__ __forceinline__ void rest_moments(T (&m)[27])
{
    using L = Lat<Q>;
    static_for<27>([&](auto ic) {
        constexpr int p = ic / 9, q = (ic / 3) % 3, r = ic % 3;
        if constexpr (L::has_moment(p, q, r) && p != 1 && q != 1 && r != 1) {
            constexpr double v = (p == 2 ? 1.0 / 3.0 : 1.0) * (q == 2 ? 1.0 / 3.0 : 1.0) * (r == 2 ? 1.0 / 3.0 : 1.0);
            m[ic] += T(SIGN * v);
        }
    });
}

// extended ("non-weighted") equilibrium: populations whose raw moments are rho prod m_p(u_a)
// (on D3Q19 the NW4 equilibrium).  Output is E_k - (SHIFT ? t_k : 0).
template <int Q, bool SHIFT, class T>
__device__ __forceinline__ void equilibrium_ext(T rho, const T (&u)[3], T (&E)[Q])
{
    using L = Lat<Q>;
    T m[27];
    static_for<27>([&](auto ic) {
        constexpr int p = ic / 9, q = (ic / 3) % 3, r = ic % 3;
        if constexpr (L::has_moment(p, q, r))
            m[ic] = rho * eq_factor<B_RAW, p>(u[0]) * eq_factor<B_RAW, q>(u[1]) * eq_factor<B_RAW, r>(u[2]);
        else m[ic] = T(0);
    });
    if constexpr (SHIFT) rest_moments<Q, -1>(m);
    pop_from_raw<Q>(m, E);
}

// ---------------------------------------------------------------- the operator
// f (or g = f - t when SHIFT) in, post-collision value out, in place.
template <int Q, int MODEL_OR_VARIANT, bool SHIFT, class T>
__device__ __forceinline__ void collide(T (&f)[Q], const Rates<T>& rt)
{
    using L = Lat<Q>;
    constexpr int MODEL = model_base(MODEL_OR_VARIANT);
    constexpr bool EQHI = model_eq_hi(MODEL_OR_VARIANT);
    T rho, drho, u[3];
    moments_rho_u<Q, SHIFT>(f, rho, drho, u);

    if constexpr (MODEL == M_BGK_W2) {
        // f_out = f - omega (f - E), pair by pair (Eq 6-7)
        const T usq15 = T(1.5) * (u[0] * u[0] + u[1] * u[1] + u[2] * u[2]);
        const T om = rt.omega, omc = T(1) - rt.omega;
        static_for<L::NH>([&](auto kc) {
            constexpr int k = kc, kb = L::opp(k);
            const T tk = T(L::w(k));
            const T cu = c_dot<Q, k>(u);
            const T quad = T(4.5) * cu * cu - usq15;
            const T sym = SHIFT ? tk * (drho + rho * quad) : tk * rho * (T(1) + quad);
            const T asym = T(3) * tk * rho * cu;
            f[k] = omc * f[k] + om * (sym + asym);
            f[kb] = omc * f[kb] + om * (sym - asym);
        });
        const T t0 = T(L::w(L::REST));
        const T e0 = SHIFT ? t0 * (drho - rho * usq15) : t0 * rho * (T(1) - usq15);
        f[L::REST] = omc * f[L::REST] + om * e0;
    } else if constexpr (MODEL == M_TRT) {
        // symmetric part relaxed with omega+, antisymmetric with omega- (R15):
        //   f_k' = f_k - w+ (fs - Es) - w- (fa - Ea),  fs = (f_k + f_kbar)/2, fa = (f_k - f_kbar)/2
        //        = a f_k + b f_kbar + (w+ Es + w- Ea),  a = 1 - (w+ + w-)/2, b = (w- - w+)/2
        const T usq15 = T(1.5) * (u[0] * u[0] + u[1] * u[1] + u[2] * u[2]);
        const T wp = rt.omega, wm = rt.omega_minus;
        const T ca = T(1) - T(0.5) * (wp + wm), cb = T(0.5) * (wm - wp);
        static_for<L::NH>([&](auto kc) {
            constexpr int k = kc, kb = L::opp(k);
            const T tk = T(L::w(k));
            const T cu = c_dot<Q, k>(u);
            const T quad = T(4.5) * cu * cu - usq15;
            const T esym = wp * (SHIFT ? tk * (drho + rho * quad) : tk * rho * (T(1) + quad));
            const T easym = wm * (T(3) * tk * rho * cu);
            const T fk = f[k], fb = f[kb];
            f[k] = ca * fk + cb * fb + (esym + easym);
            f[kb] = ca * fb + cb * fk + (esym - easym);
        });
        const T t0 = T(L::w(L::REST));
        const T e0 = SHIFT ? t0 * (drho - rho * usq15) : t0 * rho * (T(1) - usq15);
        f[L::REST] = f[L::REST] - wp * (f[L::REST] - e0);
    } else if constexpr (MODEL == M_REG) {
        // f_out = E + (1 - omega) t_k / (2 c_s^4) (c c - c_s^2 I) : Pi_neq   (R18)
        T pxx = T(0), pyy = T(0), pzz = T(0), pxy = T(0), pxz = T(0), pyz = T(0);
        static_for<L::NH>([&](auto kc) {
            constexpr int k = kc, kb = L::opp(k);
            const T sp = f[k] + f[kb];
            if constexpr (L::cx(k) != 0) pxx += sp;
            if constexpr (L::cy(k) != 0) pyy += sp;
            if constexpr (L::cz(k) != 0) pzz += sp;
            if constexpr (L::cx(k) * L::cy(k) != 0) pxy += T(L::cx(k) * L::cy(k)) * sp;
            if constexpr (L::cx(k) * L::cz(k) != 0) pxz += T(L::cx(k) * L::cz(k)) * sp;
            if constexpr (L::cy(k) * L::cz(k) != 0) pyz += T(L::cy(k) * L::cz(k)) * sp;
        });
        // subtract the second moment of E: rho (u u + c_s^2 I); with SHIFT the stored sums already
        // lack c_s^2 I, so only (rho - 1) c_s^2 I is left to remove
        const T iso = (SHIFT ? drho : rho) * T(1.0 / 3.0);
        pxx -= iso + rho * u[0] * u[0];
        pyy -= iso + rho * u[1] * u[1];
        pzz -= iso + rho * u[2] * u[2];
        pxy -= rho * u[0] * u[1];
        pxz -= rho * u[0] * u[2];
        pyz -= rho * u[1] * u[2];
        const T tr3 = (pxx + pyy + pzz) * T(1.0 / 3.0);
        const T usq15 = T(1.5) * (u[0] * u[0] + u[1] * u[1] + u[2] * u[2]);
        const T omc = T(1) - rt.omega;
        static_for<L::NH>([&](auto kc) {
            constexpr int k = kc, kb = L::opp(k);
            const T tk = T(L::w(k));
            const T cu = c_dot<Q, k>(u);
            const T quad = T(4.5) * cu * cu - usq15;
            const T esym = SHIFT ? tk * (drho + rho * quad) : tk * rho * (T(1) + quad);
            const T easym = T(3) * tk * rho * cu;
            T qp = -tr3;
            if constexpr (L::cx(k) != 0) qp += pxx;
            if constexpr (L::cy(k) != 0) qp += pyy;
            if constexpr (L::cz(k) != 0) qp += pzz;
            if constexpr (L::cx(k) * L::cy(k) != 0) qp += T(2 * L::cx(k) * L::cy(k)) * pxy;
            if constexpr (L::cx(k) * L::cz(k) != 0) qp += T(2 * L::cx(k) * L::cz(k)) * pxz;
            if constexpr (L::cy(k) * L::cz(k) != 0) qp += T(2 * L::cy(k) * L::cz(k)) * pyz;
            const T neq = omc * T(4.5) * tk * qp;  // same for k and kbar: (c c) is even in c
            f[k] = esym + easym + neq;
            f[kb] = esym - easym + neq;
        });
        const T t0 = T(L::w(L::REST));
        const T e0 = SHIFT ? t0 * (drho - rho * usq15) : t0 * rho * (T(1) - usq15);
        f[L::REST] = e0 + omc * T(4.5) * t0 * (-tr3);
    } else {
        T m[27];
        raw_from_pop<Q>(f, m);
        if constexpr (SHIFT) rest_moments<Q, +1>(m);
        if constexpr (MODEL == M_BGK_NW4) {
            // BGK towards the extended equilibrium == every raw moment relaxed with omega
            Rates<T> r1 = rt;
            r1.omega_bulk = rt.omega; r1.omega3 = rt.omega; r1.omega_hi = rt.omega;
            relax_moments<Q, B_RAW>(m, rho, u, r1);
        } else if constexpr (MODEL == M_RM) {
            relax_moments<Q, B_RAW, EQHI>(m, rho, u, rt);
        } else if constexpr (MODEL == M_HM) {
            basis_map<Q, TO_HERMITE>(m, u);
            relax_moments<Q, B_HERMITE, EQHI>(m, rho, u, rt);
            basis_map<Q, FROM_HERMITE>(m, u);
        } else if constexpr (MODEL == M_CM) {
            basis_map<Q, TO_CENTRAL>(m, u);
            relax_moments<Q, B_CENTRAL, EQHI>(m, rho, u, rt);
            basis_map<Q, FROM_CENTRAL>(m, u);
        } else if constexpr (MODEL == M_CHM) {
            basis_map<Q, TO_CENTRAL>(m, u);
            basis_map<Q, TO_HERMITE>(m, u);
            relax_moments<Q, B_CENTRAL_HERMITE, EQHI>(m, rho, u, rt);
            basis_map<Q, FROM_HERMITE>(m, u);
            basis_map<Q, FROM_CENTRAL>(m, u);
        } else if constexpr (MODEL == M_K) {
            // cumulants of the central moments per unit density; orders <= 3 coincide with them
            basis_map<Q, TO_CENTRAL>(m, u);
            const T inv = T(1) / rho;
            static_for<27>([&](auto ic) {
                if constexpr (L::has_moment(ic / 9, (ic / 3) % 3, ic % 3)) m[ic] *= inv;
            });
            cumulants_fwd<Q>(m);
            relax_moments<Q, B_CUMULANT, EQHI>(m, T(1), u, rt);
            cumulants_bwd<Q>(m);
            static_for<27>([&](auto ic) {
                if constexpr (L::has_moment(ic / 9, (ic / 3) % 3, ic % 3)) m[ic] *= rho;
            });
            basis_map<Q, FROM_CENTRAL>(m, u);
        } else if constexpr (MODEL == M_RR) {
            // Hermite space; second-order non-equilibrium moments measured, orders >= 3 rebuilt
            // from them by the recursion, in its closed form
            //   a_n = sum_a C(n_a,2) u^(n-2e_a) a_aa + sum_{a<b} n_a n_b u^(n-e_a-e_b) a_ab
            basis_map<Q, TO_HERMITE>(m, u);
            const T axx = m[18] - rho * u[0] * u[0], ayy = m[6] - rho * u[1] * u[1], azz = m[2] - rho * u[2] * u[2];
            const T axy = m[12] - rho * u[0] * u[1], axz = m[10] - rho * u[0] * u[2], ayz = m[4] - rho * u[1] * u[2];
            relax_moments<Q, B_HERMITE>(m, rho, u, rt);
            const T up[3][3] = {{T(1), u[0], u[0] * u[0]}, {T(1), u[1], u[1] * u[1]}, {T(1), u[2], u[2] * u[2]}};
            static_for<27>([&](auto ic) {
                constexpr int p = ic / 9, q = (ic / 3) % 3, r = ic % 3, order = p + q + r;
                if constexpr (order >= 3 && L::has_moment(p, q, r)) {
                    T an = T(0);
                    if constexpr (p == 2) an += up[1][q] * up[2][r] * axx;
                    if constexpr (q == 2) an += up[0][p] * up[2][r] * ayy;
                    if constexpr (r == 2) an += up[0][p] * up[1][q] * azz;
                    if constexpr (p >= 1 && q >= 1) an += T(p * q) * up[0][p - 1] * up[1][q - 1] * up[2][r] * axy;
                    if constexpr (p >= 1 && r >= 1) an += T(p * r) * up[0][p - 1] * up[1][q] * up[2][r - 1] * axz;
                    if constexpr (q >= 1 && r >= 1) an += T(q * r) * up[0][p] * up[1][q - 1] * up[2][r - 1] * ayz;
                    const T meq = rho * up[0][p] * up[1][q] * up[2][r];
                    const T w = order == 3 ? rt.omega3 : rt.omega_hi;
                    m[ic] = meq + (T(1) - w) * an;
                }
            });
            basis_map<Q, FROM_HERMITE>(m, u);
        }
        if constexpr (SHIFT) rest_moments<Q, -1>(m);
        pop_from_raw<Q>(m, f);
    }
}

}  // namespace lbm
