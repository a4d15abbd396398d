/*
 * lbm_oracle.c -- plain, slow, obviously-correct CPU oracle for the lattice
 * Boltzmann stream-and-collide update of arxiv 2010.11751 (Latt, Coreixas, Beny).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may build, load or call it.
 * It shares no code, header, table or constant generator with the CUDA path under
 * paper_2010_11751_b200/csrc/ and neither side includes or imports the other.
 *
 * What it computes (all citations are PAPER.md lines):
 *   - collide-stream cycle, Eq 1-2 (L78-83), written out as the definition:
 *       f_out_k(x,t) = Omega_k(f(x,t));   f_k(x+c_k, t+1) = f_out_k(x,t)
 *   - link-wise half-way bounce-back with momentum exchange, Eq 3 (L87-92):
 *       f_kbar(x,t+1) = f_out_k(x,t) - 6 t_k rho_w c_k.u_w,   rho_w = 1
 *   - data: AoS, two arrays, fp64 (L106, L124-126), index i = (ix*ny+iy)*nz+iz (L289-294)
 *   - collision models (L110-112, L305-352): BGK-W2 (Eq 6), BGK-NW4, TRT, RM, HM, CM,
 *     CHM, K, RR in the generic moment formulation (Eq 11-12, the slow form the paper
 *     warns about at L338 -- that is the point), bulk-viscosity mixing Eq 13-15, plus
 *     the regularised BGK that BASELINE.json config 3 asks for.
 *   - there is no blocking, fusion or reordering beyond what those equations state.
 *
 * Readings of garbled / silent passages follow SURVEY.md 8(c) R1..R24 and are listed
 * in DESIGN.md.  The ones used here: R1 (-1.5|u|^2 in Eq 6), R3 (brackets of Eq 13-15
 * are (M - M^eq)), R7 (velocity order), R8 (weights), R14 (default rates), R15 (TRT
 * magic parameter 1/4, W2 equilibrium), R16 (Eq 12 is rho*M), R17 (D3Q27 as the tensor
 * product extension), R18 (REG), R19 (kinetic energy = sum_fluid 1/2 rho |u|^2).
 *
 * Pins (tests/test_oracle_*.py): P1..P15 of SURVEY.md 8(c), P16..P18 of DESIGN.md 5.  Parity with the authors'
 * own code for RM/HM/CM/CHM/K/RR/NW4 beyond those pins is "parity unpinned": Ref [31]
 * App. G and the stlbm sources are not available.
 *
 * Build: gcc -O2 -ffp-contract=off -fopenmp -shared -fPIC (see oracle/build.py).
 */
#include <math.h>
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define QMAX 27
#define CS2 (1.0 / 3.0) /* c_s^2, L352 */

enum { O_BGK_W2 = 0, O_BGK_NW4, O_TRT, O_RM, O_HM, O_CM, O_CHM, O_K, O_RR, O_REG, O_NMODELS };
enum { B_RAW = 0, B_HERMITE, B_CENTRAL, B_CENTRAL_HERMITE };
enum { CELL_FLUID = 0, CELL_WALL = 1, CELL_MOVING = 2 };

/* ------------------------------------------------------------------ lattice */

typedef struct {
    int Q;
    int c[QMAX][3];   /* discrete velocities c_k, R7 order                     */
    int opp[QMAX];    /* kbar: c_kbar = -c_k (L92)                             */
    double t[QMAX];   /* weights t_k (R8)                                      */
    int mom[QMAX][3]; /* the moment index set I = {(p,q,r)} (Eq 8, Eq 12)      */
    int midx[3][3][3];/* (p,q,r) -> position in mom[], or -1                   */
    double Rinv[QMAX][QMAX]; /* inverse of the raw-moment matrix of Eq 12      */
} lattice_t;

static int gauss_solve(int n, const double *A, const double *b, double *x);
static int gauss_invert(int n, const double *A, double *Ainv);

/* R7: half set k=0..8 (D3Q19) / 0..12 (D3Q27), then rest, then the negatives. */
static void lattice_init(lattice_t *L, int Q)
{
    static const int half19[9][3] = {
        {-1, 0, 0}, {0, -1, 0}, {0, 0, -1}, {-1, -1, 0}, {-1, 1, 0},
        {-1, 0, -1}, {-1, 0, 1}, {0, -1, -1}, {0, -1, 1}};
    static const int extra27[4][3] = {{-1, -1, -1}, {-1, -1, 1}, {-1, 1, -1}, {-1, 1, 1}};
    int nh = (Q == 19) ? 9 : 13;
    memset(L, 0, sizeof *L);
    L->Q = Q;
    for (int k = 0; k < 9; ++k)
        for (int a = 0; a < 3; ++a) L->c[k][a] = half19[k][a];
    if (Q == 27)
        for (int k = 0; k < 4; ++k)
            for (int a = 0; a < 3; ++a) L->c[9 + k][a] = extra27[k][a];
    for (int a = 0; a < 3; ++a) L->c[nh][a] = 0;
    for (int k = 0; k < nh; ++k)
        for (int a = 0; a < 3; ++a) L->c[nh + 1 + k][a] = -L->c[k][a];
    for (int k = 0; k < Q; ++k)
        for (int j = 0; j < Q; ++j)
            if (L->c[j][0] == -L->c[k][0] && L->c[j][1] == -L->c[k][1] && L->c[j][2] == -L->c[k][2])
                L->opp[k] = j;
    /* R8: textbook weights by |c|^2 */
    for (int k = 0; k < Q; ++k) {
        int n2 = L->c[k][0] * L->c[k][0] + L->c[k][1] * L->c[k][1] + L->c[k][2] * L->c[k][2];
        if (Q == 19)
            L->t[k] = (n2 == 0) ? 1.0 / 3.0 : (n2 == 1) ? 1.0 / 18.0 : 1.0 / 36.0;
        else
            L->t[k] = (n2 == 0) ? 8.0 / 27.0 : (n2 == 1) ? 2.0 / 27.0 : (n2 == 2) ? 1.0 / 54.0 : 1.0 / 216.0;
    }
    /* moment index set: D3Q27 all of {0,1,2}^3; D3Q19 those with at least one zero index */
    int n = 0;
    for (int p = 0; p < 3; ++p)
        for (int q = 0; q < 3; ++q)
            for (int r = 0; r < 3; ++r) {
                L->midx[p][q][r] = -1;
                if (Q == 19 && p > 0 && q > 0 && r > 0) continue;
                L->mom[n][0] = p; L->mom[n][1] = q; L->mom[n][2] = r;
                L->midx[p][q][r] = n++;
            }
    /* Eq 12: R[(pqr),k] = c_kx^p c_ky^q c_kz^r, inverted numerically once */
    double R[QMAX * QMAX];
    for (int m = 0; m < Q; ++m)
        for (int k = 0; k < Q; ++k)
            R[m * Q + k] = pow(L->c[k][0], L->mom[m][0]) * pow(L->c[k][1], L->mom[m][1]) * pow(L->c[k][2], L->mom[m][2]);
    double Ri[QMAX * QMAX];
    gauss_invert(Q, R, Ri);
    for (int m = 0; m < Q; ++m)
        for (int k = 0; k < Q; ++k) L->Rinv[m][k] = Ri[m * Q + k];
}

static lattice_t g_lat19, g_lat27;
static int g_lat_ready = 0;
static const lattice_t *get_lattice(int Q)
{
#pragma omp critical(lbmo_lat)
    {
        if (!g_lat_ready) {
            lattice_init(&g_lat19, 19);
            lattice_init(&g_lat27, 27);
            g_lat_ready = 1;
        }
    }
    return Q == 19 ? &g_lat19 : Q == 27 ? &g_lat27 : NULL;
}

/* ------------------------------------------------------- dense linear algebra */

/* Gaussian elimination with partial pivoting; A is n x n row-major; returns 0 on success */
static int gauss_solve(int n, const double *A, const double *b, double *x)
{
    double M[QMAX][QMAX + 1];
    for (int i = 0; i < n; ++i) {
        for (int j = 0; j < n; ++j) M[i][j] = A[i * n + j];
        M[i][n] = b[i];
    }
    for (int col = 0; col < n; ++col) {
        int piv = col;
        for (int i = col + 1; i < n; ++i)
            if (fabs(M[i][col]) > fabs(M[piv][col])) piv = i;
        if (M[piv][col] == 0.0) return -1;
        if (piv != col)
            for (int j = 0; j <= n; ++j) { double s = M[col][j]; M[col][j] = M[piv][j]; M[piv][j] = s; }
        for (int i = col + 1; i < n; ++i) {
            double fct = M[i][col] / M[col][col];
            for (int j = col; j <= n; ++j) M[i][j] -= fct * M[col][j];
        }
    }
    for (int i = n - 1; i >= 0; --i) {
        double s = M[i][n];
        for (int j = i + 1; j < n; ++j) s -= M[i][j] * x[j];
        x[i] = s / M[i][i];
    }
    return 0;
}

static int gauss_invert(int n, const double *A, double *Ainv)
{
    double e[QMAX], col[QMAX];
    for (int j = 0; j < n; ++j) {
        for (int i = 0; i < n; ++i) e[i] = (i == j) ? 1.0 : 0.0;
        if (gauss_solve(n, A, e, col)) return -1;
        for (int i = 0; i < n; ++i) Ainv[i * n + j] = col[i];
    }
    return 0;
}

/* ---------------------------------------------------------- relaxation setup */

typedef struct {
    int model;
    double omega;      /* shear rate omega_nu, nu = (1/omega - 1/2) c_s^2 (L352)   */
    double omega_bulk; /* omega_nu_b of Eq 13-15                                   */
    double omega3;     /* rate of every moment of total order 3 (Eq 11, R14)       */
    double omega_hi;   /* rate of every moment of total order >= 4 (Eq 11, R14)    */
    double trt_magic;  /* Lambda = (1/w+ - 1/2)(1/w- - 1/2), R15                   */
    double force[3];   /* oracle-only body force for pin P4; zero otherwise        */
} relax_t;

/* R14 defaults: bulk = omega; orders >= 3 relaxed with 1, except RR whose reconstructed
 * non-equilibrium orders >= 3 are scaled by (1 - omega) like the second order. */
static void relax_defaults(relax_t *r, int model, double omega)
{
    r->model = model;
    r->omega = omega;
    r->omega_bulk = omega;
    r->omega3 = (model == O_RR) ? omega : 1.0;
    r->omega_hi = (model == O_RR) ? omega : 1.0;
    r->trt_magic = 0.25;
    r->force[0] = r->force[1] = r->force[2] = 0.0;
}

/* ------------------------------------------------------------- equilibria */

/* Eq 6 (L311) with the -1.5|u|^2 reading (R1) */
static void eq_w2(const lattice_t *L, double rho, const double u[3], double *E)
{
    double usq = u[0] * u[0] + u[1] * u[1] + u[2] * u[2];
    for (int k = 0; k < L->Q; ++k) {
        double cu = L->c[k][0] * u[0] + L->c[k][1] * u[1] + L->c[k][2] * u[2];
        E[k] = rho * L->t[k] * (1.0 + 3.0 * cu + 4.5 * cu * cu - 1.5 * usq);
    }
}

/* one-dimensional equilibrium raw moments m_0 = 1, m_1 = v, m_2 = v^2 + c_s^2 */
static double meq1d(int p, double v) { return p == 0 ? 1.0 : p == 1 ? v : v * v + CS2; }

/* extended ("non-weighted") equilibrium: f = R^-1 M^eq, M^eq_pqr = rho m_p(ux) m_q(uy) m_r(uz).
 * On D3Q19 this is the NW4 equilibrium. */
static void eq_ext(const lattice_t *L, double rho, const double u[3], double *E)
{
    double Meq[QMAX];
    for (int m = 0; m < L->Q; ++m)
        Meq[m] = rho * meq1d(L->mom[m][0], u[0]) * meq1d(L->mom[m][1], u[1]) * meq1d(L->mom[m][2], u[2]);
    for (int k = 0; k < L->Q; ++k) {
        double s = 0.0;
        for (int m = 0; m < L->Q; ++m) s += L->Rinv[k][m] * Meq[m];
        E[k] = s;
    }
}

static int model_uses_w2(int model) { return model == O_BGK_W2 || model == O_TRT || model == O_REG; }

static void eq_of_model(const lattice_t *L, int model, double rho, const double u[3], double *E)
{
    if (model_uses_w2(model)) eq_w2(L, rho, u, E);
    else eq_ext(L, rho, u, E);
}

/* ------------------------------------------------------------ moment bases */

static double hermite1d(int p, double v) { return p == 0 ? 1.0 : p == 1 ? v : v * v - CS2; }
static double power1d(int p, double v) { return p == 0 ? 1.0 : p == 1 ? v : v * v; }

/* B[(pqr),k]: raw c^p; Hermite H_p(c); central (c-u)^p; central Hermite H_p(c-u) */
static void basis_matrix(const lattice_t *L, int kind, const double u[3], double *B)
{
    int Q = L->Q;
    for (int m = 0; m < Q; ++m)
        for (int k = 0; k < Q; ++k) {
            double v = 1.0;
            for (int a = 0; a < 3; ++a) {
                double x = L->c[k][a];
                if (kind == B_CENTRAL || kind == B_CENTRAL_HERMITE) x -= u[a];
                v *= (kind == B_HERMITE || kind == B_CENTRAL_HERMITE) ? hermite1d(L->mom[m][a], x)
                                                                     : power1d(L->mom[m][a], x);
            }
            B[m * Q + k] = v;
        }
}

static void matvec(int n, const double *A, const double *x, double *y)
{
    for (int i = 0; i < n; ++i) {
        double s = 0.0;
        for (int j = 0; j < n; ++j) s += A[i * n + j] * x[j];
        y[i] = s;
    }
}

static void rho_u(const lattice_t *L, const double *f, double *rho, double u[3])
{
    double r = 0.0, j[3] = {0.0, 0.0, 0.0};
    for (int k = 0; k < L->Q; ++k) {
        r += f[k];
        for (int a = 0; a < 3; ++a) j[a] += L->c[k][a] * f[k];
    }
    *rho = r;
    for (int a = 0; a < 3; ++a) u[a] = j[a] / r;
}

static double rate_of_order(const relax_t *rx, int order)
{
    if (order <= 1) return 0.0; /* conserved: M = M^eq, not relaxed */
    if (order == 2) return rx->omega;
    if (order == 3) return rx->omega3;
    return rx->omega_hi;
}

/* Eq 11 for every moment, with Eq 13-15 (R3 reading) on the three diagonal second-order ones.
 * m, meq, mstar are in the model's own basis, ordered like L->mom. */
static void relax_moments(const lattice_t *L, const relax_t *rx, const double *m, const double *meq, double *mstar)
{
    int Q = L->Q;
    for (int i = 0; i < Q; ++i) {
        int order = L->mom[i][0] + L->mom[i][1] + L->mom[i][2];
        double w = rate_of_order(rx, order);
        mstar[i] = m[i] - w * (m[i] - meq[i]);
    }
    double wm = (rx->omega_bulk - rx->omega) / 3.0; /* omega_- (L352) */
    double wp = wm + rx->omega;                      /* omega_+ */
    int i200 = L->midx[2][0][0], i020 = L->midx[0][2][0], i002 = L->midx[0][0][2];
    double n200 = m[i200] - meq[i200], n020 = m[i020] - meq[i020], n002 = m[i002] - meq[i002];
    mstar[i200] = m[i200] - wp * n200 - wm * n020 - wm * n002; /* Eq 13 */
    mstar[i020] = m[i020] - wm * n200 - wp * n020 - wm * n002; /* Eq 14 */
    mstar[i002] = m[i002] - wm * n200 - wm * n020 - wp * n002; /* Eq 15 */
}

/* ----------------------------------------------------- cumulants (model K) */

static double binom2(int n, int k) /* n <= 2 */
{
    static const double b[3][3] = {{1, 0, 0}, {1, 1, 0}, {1, 2, 1}};
    return b[n][k];
}

/* General moment <-> cumulant relation from M(t) = exp(K(t)), d_i M = (d_i K) M, by Leibniz:
 *   m_n = sum_{0 <= k <= n - e_i} C(n - e_i, k) K_{k + e_i} m_{n - e_i - k},   m_0 = 1,
 * for any axis i with n_i >= 1.  dir = +1: fill K from m;  dir = -1: fill m from K.
 * All lower multi-indices needed exist in the D3Q19 set because it is a lower set. */
static void moment_cumulant(const lattice_t *L, int dir, double *m, double *K)
{
    int Q = L->Q;
    for (int order = 1; order <= 6; ++order)
        for (int idx = 0; idx < Q; ++idx) {
            const int *n = L->mom[idx];
            if (n[0] + n[1] + n[2] != order) continue;
            int i = n[0] > 0 ? 0 : n[1] > 0 ? 1 : 2;
            int np[3] = {n[0], n[1], n[2]};
            np[i] -= 1;
            double s = 0.0;
            for (int a = 0; a <= np[0]; ++a)
                for (int b = 0; b <= np[1]; ++b)
                    for (int c = 0; c <= np[2]; ++c) {
                        if (a == np[0] && b == np[1] && c == np[2]) continue; /* the K_n m_0 term */
                        int kk[3] = {a, b, c};
                        kk[i] += 1;
                        int iK = L->midx[kk[0]][kk[1]][kk[2]];
                        int iM = L->midx[np[0] - a][np[1] - b][np[2] - c];
                        s += binom2(np[0], a) * binom2(np[1], b) * binom2(np[2], c) * K[iK] * m[iM];
                    }
            if (dir > 0) K[idx] = m[idx] - s;
            else m[idx] = K[idx] + s;
        }
}

/* --------------------------------------------- recursive regularisation (RR) */

/* a^neq_{a1..an} = u_{an} a^neq_{a1..a(n-1)} + sum_{i<n} (prod_{j != i, j<n} u_{aj}) a^neq_{ai an}
 * (the recursion L474 refers to), literal recursion over the index list. */
static double rr_recursive(const int *alpha, int n, const double u[3], const double a2[3][3])
{
    if (n == 2) return a2[alpha[0]][alpha[1]];
    double s = u[alpha[n - 1]] * rr_recursive(alpha, n - 1, u, a2);
    for (int i = 0; i < n - 1; ++i) {
        double prod = 1.0;
        for (int j = 0; j < n - 1; ++j)
            if (j != i) prod *= u[alpha[j]];
        s += prod * a2[alpha[i]][alpha[n - 1]];
    }
    return s;
}

/* ------------------------------------------------------------- collision */

static void collide(const lattice_t *L, const relax_t *rx, const double *f, double *fout)
{
    int Q = L->Q;
    double rho, u[3];
    rho_u(L, f, &rho, u); /* L180-186, L309 */
    double E[QMAX];

    switch (rx->model) {
    case O_BGK_W2: /* f - omega (f - E), Eq 6 equilibrium */
        eq_w2(L, rho, u, E);
        for (int k = 0; k < Q; ++k) fout[k] = f[k] - rx->omega * (f[k] - E[k]);
        break;
    case O_BGK_NW4: /* same with the extended equilibrium */
        eq_ext(L, rho, u, E);
        for (int k = 0; k < Q; ++k) fout[k] = f[k] - rx->omega * (f[k] - E[k]);
        break;
    case O_TRT: { /* two relaxation times on the symmetric / antisymmetric parts (R15) */
        eq_w2(L, rho, u, E);
        double wp = rx->omega;
        double wm = 1.0 / (rx->trt_magic / (1.0 / wp - 0.5) + 0.5);
        for (int k = 0; k < Q; ++k) {
            int kb = L->opp[k];
            double fp = 0.5 * (f[k] + f[kb]), fm = 0.5 * (f[k] - f[kb]);
            double ep = 0.5 * (E[k] + E[kb]), em = 0.5 * (E[k] - E[kb]);
            fout[k] = f[k] - wp * (fp - ep) - wm * (fm - em);
        }
        break;
    }
    case O_REG: { /* regularised BGK (R18): f = E + (1-omega) t_k/(2 cs^4) Q_k : Pi^neq */
        eq_w2(L, rho, u, E);
        double Pi[3][3] = {{0}};
        for (int k = 0; k < Q; ++k)
            for (int a = 0; a < 3; ++a)
                for (int b = 0; b < 3; ++b) Pi[a][b] += L->c[k][a] * L->c[k][b] * (f[k] - E[k]);
        for (int k = 0; k < Q; ++k) {
            double qp = 0.0;
            for (int a = 0; a < 3; ++a)
                for (int b = 0; b < 3; ++b)
                    qp += (L->c[k][a] * L->c[k][b] - (a == b ? CS2 : 0.0)) * Pi[a][b];
            fout[k] = E[k] + (1.0 - rx->omega) * L->t[k] / (2.0 * CS2 * CS2) * qp;
        }
        break;
    }
    case O_RM: case O_HM: case O_CM: case O_CHM: { /* m = B f; Eq 11/13-15; f = B^-1 m* */
        int kind = rx->model == O_RM ? B_RAW : rx->model == O_HM ? B_HERMITE
                 : rx->model == O_CM ? B_CENTRAL : B_CENTRAL_HERMITE;
        double B[QMAX * QMAX], m[QMAX], meq[QMAX], ms[QMAX];
        basis_matrix(L, kind, u, B);
        eq_ext(L, rho, u, E);
        matvec(Q, B, f, m);
        matvec(Q, B, E, meq);
        relax_moments(L, rx, m, meq, ms);
        gauss_solve(Q, B, ms, fout);
        break;
    }
    case O_K: { /* cumulants of the central moments per unit density */
        double B[QMAX * QMAX], m[QMAX], kap[QMAX], K[QMAX], Keq[QMAX], Ks[QMAX], ms[QMAX];
        basis_matrix(L, B_CENTRAL, u, B);
        matvec(Q, B, f, m);
        for (int i = 0; i < Q; ++i) kap[i] = m[i] / rho;
        K[L->midx[0][0][0]] = 0.0;
        moment_cumulant(L, +1, kap, K);
        for (int i = 0; i < Q; ++i) Keq[i] = 0.0;
        Keq[L->midx[2][0][0]] = Keq[L->midx[0][2][0]] = Keq[L->midx[0][0][2]] = CS2;
        relax_moments(L, rx, K, Keq, Ks);
        ms[L->midx[0][0][0]] = 1.0;
        moment_cumulant(L, -1, ms, Ks);
        for (int i = 0; i < Q; ++i) ms[i] *= rho;
        gauss_solve(Q, B, ms, fout);
        break;
    }
    case O_RR: { /* Hermite space; orders >= 3 of the non-equilibrium part rebuilt by recursion */
        double B[QMAX * QMAX], m[QMAX], meq[QMAX], ms[QMAX];
        basis_matrix(L, B_HERMITE, u, B);
        eq_ext(L, rho, u, E);
        matvec(Q, B, f, m);
        matvec(Q, B, E, meq);
        relax_moments(L, rx, m, meq, ms); /* orders <= 2 as for HM */
        double a2[3][3];
        for (int a = 0; a < 3; ++a)
            for (int b = 0; b < 3; ++b) {
                int pq[3] = {0, 0, 0};
                pq[a] += 1; pq[b] += 1;
                int i = L->midx[pq[0]][pq[1]][pq[2]];
                a2[a][b] = m[i] - meq[i];
            }
        for (int i = 0; i < Q; ++i) {
            int order = L->mom[i][0] + L->mom[i][1] + L->mom[i][2];
            if (order < 3) continue;
            int alpha[6], n = 0;
            for (int a = 0; a < 3; ++a)
                for (int r = 0; r < L->mom[i][a]; ++r) alpha[n++] = a;
            double an = rr_recursive(alpha, n, u, a2);
            ms[i] = meq[i] + (1.0 - rate_of_order(rx, order)) * an;
        }
        gauss_solve(Q, B, ms, fout);
        break;
    }
    default:
        for (int k = 0; k < Q; ++k) fout[k] = NAN;
    }
    /* oracle-only constant body force (pin P4): f_out_k += 3 t_k rho c_k.g */
    if (rx->force[0] != 0.0 || rx->force[1] != 0.0 || rx->force[2] != 0.0)
        for (int k = 0; k < Q; ++k)
            fout[k] += 3.0 * L->t[k] * rho *
                       (L->c[k][0] * rx->force[0] + L->c[k][1] * rx->force[1] + L->c[k][2] * rx->force[2]);
}

/* ------------------------------------------------------------- simulation */

typedef struct lbmo_ctx {
    const lattice_t *L;
    int nx, ny, nz;
    size_t N;
    relax_t rx;
    uint8_t *flags;  /* [N] */
    double u_wall[3];
    double *f;       /* [N][Q] pre-collision populations at the current time */
    double *fnew;    /* [N][Q] */
    long steps;
} lbmo_t;

static int wrap(int i, int n) { return i < 0 ? i + n : i >= n ? i - n : i; }

lbmo_t *lbmo_create(int nx, int ny, int nz, int Q, int model, double omega)
{
    const lattice_t *L = get_lattice(Q);
    if (!L || nx < 1 || ny < 1 || nz < 1 || model < 0 || model >= O_NMODELS) return NULL;
    lbmo_t *o = (lbmo_t *)calloc(1, sizeof *o);
    o->L = L; o->nx = nx; o->ny = ny; o->nz = nz;
    o->N = (size_t)nx * ny * nz;
    relax_defaults(&o->rx, model, omega);
    o->flags = (uint8_t *)calloc(o->N, 1);
    o->f = (double *)calloc(o->N * Q, sizeof(double));
    o->fnew = (double *)calloc(o->N * Q, sizeof(double));
    if (!o->flags || !o->f || !o->fnew) { free(o->flags); free(o->f); free(o->fnew); free(o); return NULL; }
    return o;
}

void lbmo_destroy(lbmo_t *o)
{
    if (!o) return;
    free(o->flags); free(o->f); free(o->fnew); free(o);
}

int lbmo_set_flags(lbmo_t *o, const uint8_t *flags, const double u_wall[3])
{
    memcpy(o->flags, flags, o->N);
    for (int a = 0; a < 3; ++a) o->u_wall[a] = u_wall ? u_wall[a] : 0.0;
    return 0;
}

int lbmo_set_relaxation(lbmo_t *o, double omega_bulk, double omega3, double omega_hi)
{
    o->rx.omega_bulk = omega_bulk; o->rx.omega3 = omega3; o->rx.omega_hi = omega_hi;
    return 0;
}

int lbmo_set_trt_magic(lbmo_t *o, double lambda) { o->rx.trt_magic = lambda; return 0; }

int lbmo_set_force(lbmo_t *o, const double g[3])
{
    for (int a = 0; a < 3; ++a) o->rx.force[a] = g[a];
    return 0;
}

/* the model's own equilibrium on fluid cells, zero elsewhere */
int lbmo_init_equilibrium(lbmo_t *o, const double *rho, const double *u /* [3][N] */)
{
    int Q = o->L->Q;
    for (size_t i = 0; i < o->N; ++i) {
        double *fi = o->f + i * Q;
        if (o->flags[i] != CELL_FLUID) { for (int k = 0; k < Q; ++k) fi[k] = 0.0; continue; }
        double ui[3] = {u[i], u[o->N + i], u[2 * o->N + i]};
        eq_of_model(o->L, o->rx.model, rho[i], ui, fi);
    }
    memset(o->fnew, 0, o->N * Q * sizeof(double));
    o->steps = 0;
    return 0;
}

/* one time step: Eq 1 on every fluid cell, then Eq 2 or Eq 3 per link */
static void step_once(lbmo_t *o)
{
    const lattice_t *L = o->L;
    int Q = L->Q, nx = o->nx, ny = o->ny, nz = o->nz;
#pragma omp parallel for schedule(static)
    for (int ix = 0; ix < nx; ++ix)
        for (int iy = 0; iy < ny; ++iy)
            for (int iz = 0; iz < nz; ++iz) {
                size_t i = ((size_t)ix * ny + iy) * nz + iz;
                if (o->flags[i] != CELL_FLUID) continue;
                double fout[QMAX];
                collide(L, &o->rx, o->f + i * Q, fout);
                for (int k = 0; k < Q; ++k) {
                    int jx = wrap(ix + L->c[k][0], nx), jy = wrap(iy + L->c[k][1], ny), jz = wrap(iz + L->c[k][2], nz);
                    size_t n = ((size_t)jx * ny + jy) * nz + jz;
                    if (o->flags[n] == CELL_FLUID) {
                        o->fnew[n * Q + k] = fout[k]; /* Eq 2 */
                    } else {
                        double cuw = 0.0;
                        if (o->flags[n] == CELL_MOVING)
                            for (int a = 0; a < 3; ++a) cuw += L->c[k][a] * o->u_wall[a];
                        o->fnew[i * Q + L->opp[k]] = fout[k] - 6.0 * L->t[k] * 1.0 * cuw; /* Eq 3, rho_w = 1 */
                    }
                }
            }
    double *tmp = o->f; o->f = o->fnew; o->fnew = tmp;
    o->steps++;
}

int lbmo_step(lbmo_t *o, int n)
{
    for (int s = 0; s < n; ++s) step_once(o);
    return 0;
}

/* populations in [Q][N] order, zero on non-fluid cells */
int lbmo_get_populations(const lbmo_t *o, double *f)
{
    int Q = o->L->Q;
    for (size_t i = 0; i < o->N; ++i)
        for (int k = 0; k < Q; ++k)
            f[(size_t)k * o->N + i] = (o->flags[i] == CELL_FLUID) ? o->f[i * Q + k] : 0.0;
    return 0;
}

int lbmo_set_populations(lbmo_t *o, const double *f)
{
    int Q = o->L->Q;
    for (size_t i = 0; i < o->N; ++i)
        for (int k = 0; k < Q; ++k)
            o->f[i * Q + k] = (o->flags[i] == CELL_FLUID) ? f[(size_t)k * o->N + i] : 0.0;
    return 0;
}

/* rho and u = sum c f / rho (+ g/2 with the oracle-only force), zero on non-fluid cells */
int lbmo_macroscopic(const lbmo_t *o, double *rho, double *u /* [3][N] */)
{
    for (size_t i = 0; i < o->N; ++i) {
        double r = 0.0, ui[3] = {0.0, 0.0, 0.0};
        if (o->flags[i] == CELL_FLUID) {
            rho_u(o->L, o->f + i * o->L->Q, &r, ui);
            for (int a = 0; a < 3; ++a) ui[a] += 0.5 * o->rx.force[a];
        }
        rho[i] = r;
        for (int a = 0; a < 3; ++a) u[a * o->N + i] = ui[a];
    }
    return 0;
}

/* R19: E = sum over fluid cells of 1/2 rho |u|^2, long double accumulation */
int lbmo_kinetic_energy(const lbmo_t *o, double *e)
{
    long double acc = 0.0L;
    for (size_t i = 0; i < o->N; ++i) {
        if (o->flags[i] != CELL_FLUID) continue;
        double r, ui[3];
        rho_u(o->L, o->f + i * o->L->Q, &r, ui);
        acc += 0.5L * (long double)r * ((long double)ui[0] * ui[0] + (long double)ui[1] * ui[1] + (long double)ui[2] * ui[2]);
    }
    *e = (double)acc;
    return 0;
}

long lbmo_steps(const lbmo_t *o) { return o->steps; }

int lbmo_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ------------------------------------------- single-cell entry points (pins) */

int lbmo_lattice(int Q, int *c /* [Q][3] */, double *t, int *opp, int *mom /* [Q][3] */)
{
    const lattice_t *L = get_lattice(Q);
    if (!L) return -1;
    for (int k = 0; k < Q; ++k) {
        for (int a = 0; a < 3; ++a) { c[3 * k + a] = L->c[k][a]; mom[3 * k + a] = L->mom[k][a]; }
        t[k] = L->t[k];
        opp[k] = L->opp[k];
    }
    return 0;
}

/* kind 0: Eq 6 (W2); kind 1: extended / NW4 */
int lbmo_equilibrium(int Q, int kind, double rho, const double u[3], double *E)
{
    const lattice_t *L = get_lattice(Q);
    if (!L) return -1;
    if (kind == 0) eq_w2(L, rho, u, E);
    else eq_ext(L, rho, u, E);
    return 0;
}

/* rates[5] = {omega, omega_bulk, omega3, omega_hi, trt_magic}; a NaN entry keeps the default */
int lbmo_collide(int Q, int model, const double *rates, const double *f, double *fout)
{
    const lattice_t *L = get_lattice(Q);
    if (!L || model < 0 || model >= O_NMODELS) return -1;
    relax_t rx;
    relax_defaults(&rx, model, rates[0]);
    if (!isnan(rates[1])) rx.omega_bulk = rates[1];
    if (!isnan(rates[2])) rx.omega3 = rates[2];
    if (!isnan(rates[3])) rx.omega_hi = rates[3];
    if (!isnan(rates[4])) rx.trt_magic = rates[4];
    collide(L, &rx, f, fout);
    return 0;
}

/* moments of f in one of the four bases, about the velocity u (ignored for raw / Hermite) */
int lbmo_moments(int Q, int kind, const double u[3], const double *f, double *m)
{
    const lattice_t *L = get_lattice(Q);
    if (!L) return -1;
    double B[QMAX * QMAX];
    basis_matrix(L, kind, u, B);
    matvec(Q, B, f, m);
    return 0;
}

/* cumulants of normalised central moments kap (kap_000 = 1), ordered like the moment set */
int lbmo_cumulants(int Q, int dir, double *kap, double *K)
{
    const lattice_t *L = get_lattice(Q);
    if (!L) return -1;
    moment_cumulant(L, dir, kap, K);
    return 0;
}
