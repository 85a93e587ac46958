/*
 * acm_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, unfused CPU implementation (fp64) of the per-time-step coupled
 * lattice-Boltzmann update of the conservative Allen-Cahn model of
 * arXiv 2012.06144 (PAPER.md, "P:<line>" below), written from the paper's
 * equations in the paper's order and notation.  It is the oracle the CUDA path
 * is checked against.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference leg may build, load or call it.  It shares no
 * code, header, table or constant generator with paper_2012_06144_b200/csrc.
 *
 * Structure: separate full-grid passes (P1..P5 phase-field LB step, H1..H6
 * hydrodynamic LB step), explicit moment matrices M, M^-1 and diagonal
 * relaxation matrices S, i.e. Omega = M^-1 S M applied literally (eq. 25
 * P:215-231).  No blocking, no fusion, no closed-form collision.
 *
 * Readings of the paper where it is silent/garbled (ids
 * A1..A19 follow SURVEY.md section 8(c-2)):
 *   A1  theta = (1 - 4 (phi-phi0)^2) / xi
 *   A2  omega_phi = 1/(tau_phi + 1/2), tau_phi = M/c_s^2
 *   A3  phase collision: MRT, first-order moments at omega_phi, others at 1,
 *       weighted-orthogonal moment basis
 *   A4  hydro collision: all six second-order moments at s_nu, others at 1
 *   A6  eq. 25 taken from the listing P:229: m - (m - meq + F_m/2) S + F_m
 *   A7  grad phi as opposite-pair differences; n = 0 where |grad phi| == 0
 *   A8  eqs. 23-24 use the stencil of the LB step that evaluates them
 *   A9  eq. 18: F_mu,a = -(nu/c_s^2) sum_b [sum_k e_ka e_kb (Omega(g-geq))_k] d_b rho
 *   A10 geq inside F_mu uses u of the previous hydro step (single evaluation)
 *   A11 h^eq uses phi_new = sum of the streamed h; theta, n use the previous phi
 *   A12 phase step first (with u of the previous step), then hydro with new phi
 *   A13 phase = stream(pull) then collide; hydro = collide then stream(push)
 *   A14 init: h = phi Gamma(u), g = Gamma(u) - w (p* = 0)
 *   A15 grad rho = (rho_H - rho_L) grad phi
 *   A16 walls: half-way bounce-back for h and g; phi ghost = mirror
 *   A17 F_b = rho(phi) * gravity (no hydrostatic subtraction)
 *   A18 no clamp on phi or rho
 *   A19 p = p* rho c_s^2
 *   A23 variant ORACLE_VAR_PHASE_SRT: Omega^h = omega_phi I
 *   A24 bubble volume/centroid/velocity over phi < 1/2, weighted with 1 - phi
 *   A25 two-dimensional instance: D2Q9 for both LB steps on one plane
 *   A26 variant ORACLE_VAR_BULK_ONE: the trace of the second-order moments ("bulk" moment
 *       x^2+y^2+z^2) counts among "all other moments" and relaxes with 1; the five deviatoric
 *       second-order moments keep s_nu (the other reading of P:152-156, cf. A4)
 *   A27 variant oracle_set_subiter(k): eq. 22 is implicit in F_mu (P:158 with eq. 18);
 *       k fixed-point sweeps u <- sum g e + F(u)/(2 rho), F_mu re-evaluated with g^eq(u);
 *       k = 1 is reading A10
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): lattice identities, weighted
 * orthogonality of M, eq.25 forcing identity, brute-force 4^3 step against a
 * hand-expanded projector form, FD operators on polynomials, sum(phi)
 * conservation, uniform state, Galilean invariance, planar tanh profile
 * (eq. 3) and its advection with a uniform flow (eq. 1), mobility and viscosity decay rates, Poiseuille profile,
 * Laplace law;
 * variants (tests/test_oracle_variants.py, test_oracle_d2q9.py): SRT brute force and omega = 1
 * special case, bubble diagnostics (symmetry, translation, continuum volume), eqs. 31-35
 * round trip, D2Q9 lattice identities / brute force / transport limits; A26: brute force with the
 * projector split into deviatoric and trace parts, identical to the default at s_nu = 1, shear
 * viscosity unchanged, sound attenuation changed as the bulk viscosity predicts; A27: k = 1 is the
 * default bit for bit, the converged u satisfies eq. 22 to rounding (residual from a brute-force F).
 * Two-phase flow: layered Poiseuille (F_mu) and two-layer hydrostatics (F_p), test_oracle_twophase.py.
 * Unpinned: rising-bubble drag/shape (eqs. 31-35; data only in figures).
 *
 * Build: gcc -O2 -ffp-contract=off -fopenmp -shared -fPIC (oracle/build.py).
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#include <stddef.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define QMAX 27
#define CS2 (1.0 / 3.0)          /* c_s^2, c = dx/dt = 1 */
#define PHI_L 0.0
#define PHI_H 1.0
#define PHI_0 0.5                /* (phi_L + phi_H)/2 */

enum { WALL_X = 1, WALL_Y = 2, WALL_Z = 4 };

/* ---- canonical direction list; opposite of odd k is k+1 ---- */
static const int DIRS27[27][3] = {
    {0, 0, 0},
    {1, 0, 0}, {-1, 0, 0}, {0, 1, 0}, {0, -1, 0}, {0, 0, 1}, {0, 0, -1},
    {1, 1, 0}, {-1, -1, 0}, {1, -1, 0}, {-1, 1, 0},
    {1, 0, 1}, {-1, 0, -1}, {1, 0, -1}, {-1, 0, 1},
    {0, 1, 1}, {0, -1, -1}, {0, 1, -1}, {0, -1, 1},
    {1, 1, 1}, {-1, -1, -1}, {1, 1, -1}, {-1, -1, 1},
    {1, -1, 1}, {-1, 1, -1}, {-1, 1, 1}, {1, -1, -1}};

#define ORDER_BULK 20            /* row generated by x^2+y^2+z^2 when the bulk moment is split off (A26) */

typedef struct {
    int Q;
    int e[QMAX][3];
    double w[QMAX];
    int opp[QMAX];
    double M[QMAX * QMAX];    /* moment matrix, row k = k-th moment */
    double Minv[QMAX * QMAX];
    int order[QMAX];          /* polynomial order of row k */
} lattice_t;

typedef struct oracle_ctx {
    int nx, ny, nz;
    size_t N;
    lattice_t Lh, Lg;
    double rho_H, rho_L, sigma, xi, Mob, nu_H, nu_L, grav[3];
    unsigned walls;
    double omega_phi, beta, kappa, tau_H, tau_L;
    double *H, *H2, *G, *G2, *C, *C2, *U, *U2, *tmp;
    int initialised;
    unsigned variant;         /* ORACLE_VAR_* */
    int subiter;              /* sweeps of the fixed point of eq. 22 (A27); 1 = reading A10 */
} oracle_ctx;

/* Variants of the operators the paper itself uses elsewhere:
 *   ORACLE_VAR_PHASE_SRT  single-relaxation-time phase-field collision, Omega^h = omega_phi I
 *                         ("a D3Q15 SRT LB scheme for the interface tracking"), reading A23
 *   ORACLE_VAR_BULK_ONE   hydrodynamic collision: the bulk moment (trace of the second-order moments)
 *                         relaxes with 1 like the higher moments, only the deviatoric second-order
 *                         moments with s_nu ("all other moments are relaxed by one"), reading A26 */
enum { ORACLE_VAR_PHASE_SRT = 1, ORACLE_VAR_BULK_ONE = 2 };

/* ------------------------------------------------------------------------- */
/* Lattices and moment matrices                                               */
/* ------------------------------------------------------------------------- */

static int build_stencil(int Q, lattice_t *L)
{
    /* textbook lattices named by the paper */
    int n = 0;
    memset(L, 0, sizeof(*L));
    L->Q = Q;
    for (int k = 0; k < 27; ++k) {
        int s = abs(DIRS27[k][0]) + abs(DIRS27[k][1]) + abs(DIRS27[k][2]); /* 0 rest,1 axis,2 edge,3 corner */
        double w = -1.0;
        if (Q == 9) {
            /* D2Q9: the nine directions of the x-y plane; the grid then has nz = 1 */
            if (DIRS27[k][2] != 0) continue;
            if (s == 0) w = 4.0 / 9.0; else if (s == 1) w = 1.0 / 9.0; else w = 1.0 / 36.0;
        } else if (Q == 15) {
            if (s == 0) w = 2.0 / 9.0; else if (s == 1) w = 1.0 / 9.0; else if (s == 3) w = 1.0 / 72.0;
        } else if (Q == 19) {
            if (s == 0) w = 1.0 / 3.0; else if (s == 1) w = 1.0 / 18.0; else if (s == 2) w = 1.0 / 36.0;
        } else if (Q == 27) {
            if (s == 0) w = 8.0 / 27.0; else if (s == 1) w = 2.0 / 27.0; else if (s == 2) w = 1.0 / 54.0; else w = 1.0 / 216.0;
        } else {
            return -1;
        }
        if (w < 0.0) continue;
        L->e[n][0] = DIRS27[k][0]; L->e[n][1] = DIRS27[k][1]; L->e[n][2] = DIRS27[k][2];
        L->w[n] = w;
        ++n;
    }
    if (n != Q) return -1;
    L->opp[0] = 0;
    for (int i = 1; i < Q; i += 2) { L->opp[i] = i + 1; L->opp[i + 1] = i; }
    return 0;
}

static double ipow(int b, int p) { double r = 1.0; for (int k = 0; k < p; ++k) r *= (double)b; return r; }

/* Weighted Gram-Schmidt of the monomials x^a y^b z^c (a,b,c in 0..2), taken in
 * order of total degree; <p,q> = sum_i w_i p_i q_i ("weighted orthogonal moment
 * set").  Dependent monomials are dropped.  order[k] = degree of the
 * monomial that generated row k. */
/* bulk_split (A26): among the polynomials of degree 2 the trace x^2+y^2+z^2 is taken FIRST (row order
 * ORDER_BULK); the monomials that follow then yield the deviatoric moments (the last one is dependent
 * and dropped), all of them weighted-orthogonal to the bulk row. */
static int build_moments(lattice_t *L, int bulk_split)
{
    const int Q = L->Q;
    int rows = 0;
    memset(L->M, 0, sizeof(L->M));
    for (int deg = 0; deg <= 6 && rows < Q; ++deg)
        for (int a = (bulk_split && deg == 2) ? 3 : 2; a >= 0; --a)      /* a == 3 stands for the trace */
            for (int b = 2; b >= 0; --b)
                for (int c = 2; c >= 0; --c) {
                    const int trace = (a == 3);
                    if (trace && (b != 2 || c != 2)) continue;       /* one pass for the trace generator */
                    if ((!trace && a + b + c != deg) || rows >= Q) continue;
                    double v[QMAX];
                    for (int i = 0; i < Q; ++i)
                        v[i] = trace ? (double)(L->e[i][0] * L->e[i][0] + L->e[i][1] * L->e[i][1] + L->e[i][2] * L->e[i][2])
                                     : ipow(L->e[i][0], a) * ipow(L->e[i][1], b) * ipow(L->e[i][2], c);
                    /* two passes of Gram-Schmidt for numerical cleanliness */
                    for (int pass = 0; pass < 2; ++pass)
                        for (int r = 0; r < rows; ++r) {
                            double num = 0.0, den = 0.0;
                            for (int i = 0; i < Q; ++i) {
                                num += L->w[i] * v[i] * L->M[r * Q + i];
                                den += L->w[i] * L->M[r * Q + i] * L->M[r * Q + i];
                            }
                            double f = num / den;
                            for (int i = 0; i < Q; ++i) v[i] -= f * L->M[r * Q + i];
                        }
                    double nrm = 0.0;
                    for (int i = 0; i < Q; ++i) nrm += L->w[i] * v[i] * v[i];
                    if (nrm < 1e-12) continue;          /* linearly dependent on the lattice */
                    for (int i = 0; i < Q; ++i) L->M[rows * Q + i] = v[i];
                    L->order[rows] = trace ? ORDER_BULK : deg;
                    ++rows;
                }
    if (rows != Q) return -1;

    /* M^-1 by Gauss-Jordan elimination with partial pivoting */
    double A[QMAX][2 * QMAX];
    for (int r = 0; r < Q; ++r)
        for (int c = 0; c < Q; ++c) { A[r][c] = L->M[r * Q + c]; A[r][Q + c] = (r == c) ? 1.0 : 0.0; }
    for (int col = 0; col < Q; ++col) {
        int piv = col;
        for (int r = col + 1; r < Q; ++r) if (fabs(A[r][col]) > fabs(A[piv][col])) piv = r;
        if (fabs(A[piv][col]) < 1e-14) return -1;
        if (piv != col) for (int c = 0; c < 2 * Q; ++c) { double t = A[piv][c]; A[piv][c] = A[col][c]; A[col][c] = t; }
        double d = A[col][col];
        for (int c = 0; c < 2 * Q; ++c) A[col][c] /= d;
        for (int r = 0; r < Q; ++r) {
            if (r == col) continue;
            double f = A[r][col];
            if (f == 0.0) continue;
            for (int c = 0; c < 2 * Q; ++c) A[r][c] -= f * A[col][c];
        }
    }
    for (int r = 0; r < Q; ++r) for (int c = 0; c < Q; ++c) L->Minv[r * Q + c] = A[r][Q + c];
    return 0;
}

static int build_lattice(int Q, lattice_t *L, int bulk_split)
{
    if (build_stencil(Q, L)) return -1;
    return build_moments(L, bulk_split);
}

/* Gamma_i(u), eq. 6 */
static double Gamma(const lattice_t *L, int i, const double u[3])
{
    double eu = L->e[i][0] * u[0] + L->e[i][1] * u[1] + L->e[i][2] * u[2];
    double uu = u[0] * u[0] + u[1] * u[1] + u[2] * u[2];
    return L->w[i] * (1.0 + eu / CS2 + (eu * eu) / (2.0 * CS2 * CS2) - uu / (2.0 * CS2));
}

/* y = A x, A is Q x Q row-major.  Each y[r] is accumulated over c = 0..Q-1 in
 * that order; the loops are nested column-outer only so that the Q sums advance
 * independently (no change to any sum's order of operations). */
static void matvec(int Q, const double *A, const double *x, double *y)
{
    for (int r = 0; r < Q; ++r) y[r] = 0.0;
    for (int c = 0; c < Q; ++c) {
        const double xc = x[c];
        for (int r = 0; r < Q; ++r) y[r] += A[r * Q + c] * xc;
    }
}

/* ------------------------------------------------------------------------- */
/* Geometry helpers                                                            */
/* ------------------------------------------------------------------------- */

static size_t cell(const oracle_ctx *o, int x, int y, int z)
{
    return ((size_t)z * o->ny + y) * o->nx + x;
}

/* neighbour x+d along one axis of length n: returns 1 if beyond a wall (and
 * leaves *out untouched), else wraps periodically */
static int shift(int x, int d, int n, int wall, int *out)
{
    int t = x + d;
    if (t < 0 || t >= n) {
        if (wall) return 1;
        t = (t + n) % n;
    }
    *out = t;
    return 0;
}

/* index of x + s*e; returns 1 if that cell is beyond a wall */
static int neighbour(const oracle_ctx *o, int x, int y, int z, const int e[3], int s, size_t *idx)
{
    int X, Y, Z;
    if (shift(x, s * e[0], o->nx, o->walls & WALL_X, &X)) return 1;
    if (shift(y, s * e[1], o->ny, o->walls & WALL_Y, &Y)) return 1;
    if (shift(z, s * e[2], o->nz, o->walls & WALL_Z, &Z)) return 1;
    *idx = cell(o, X, Y, Z);
    return 0;
}

/* phi at x + s*e with periodic wrap and, at walls, mirror ghost (A16):
 * C(x,-1,z) = C(x,0,z), i.e. the out-of-range coordinate is clamped */
static double phi_at(const oracle_ctx *o, const double *C, int x, int y, int z, const int e[3], int s)
{
    int c[3] = {x + s * e[0], y + s * e[1], z + s * e[2]};
    const int n[3] = {o->nx, o->ny, o->nz};
    const unsigned wl[3] = {WALL_X, WALL_Y, WALL_Z};
    for (int a = 0; a < 3; ++a) {
        if (c[a] < 0) c[a] = (o->walls & wl[a]) ? 0 : c[a] + n[a];
        else if (c[a] >= n[a]) c[a] = (o->walls & wl[a]) ? n[a] - 1 : c[a] - n[a];
    }
    return C[cell(o, c[0], c[1], c[2])];
}

/* eq. 23 with c = dx = 1:  grad phi = (1/c_s^2) sum_i e_i w_i phi(x+e_i),
 * summed as opposite-pair differences (A7) */
static void grad_phi(const oracle_ctx *o, const lattice_t *L, const double *C, int x, int y, int z, double g[3])
{
    g[0] = g[1] = g[2] = 0.0;
    for (int i = 1; i < L->Q; i += 2) {
        double d = phi_at(o, C, x, y, z, L->e[i], +1) - phi_at(o, C, x, y, z, L->e[i], -1);
        for (int a = 0; a < 3; ++a) g[a] += L->w[i] * L->e[i][a] * d;
    }
    for (int a = 0; a < 3; ++a) g[a] *= 1.0 / CS2;
}

/* eq. 24: lap phi = (2/c_s^2) sum_i w_i [phi(x+e_i) - phi(x)] */
static double lap_phi(const oracle_ctx *o, const lattice_t *L, const double *C, int x, int y, int z)
{
    const int zero[3] = {0, 0, 0};
    double c0 = phi_at(o, C, x, y, z, zero, 0), s = 0.0;
    for (int i = 1; i < L->Q; ++i) s += L->w[i] * (phi_at(o, C, x, y, z, L->e[i], +1) - c0);
    return (2.0 / CS2) * s;
}

/* ------------------------------------------------------------------------- */
/* Phase-field LB step (Alg. 2 lines 3-6): stream-pull, phi, collide    */
/* ------------------------------------------------------------------------- */

static void phase_step(oracle_ctx *o)
{
    const lattice_t *L = &o->Lh;
    const int Q = L->Q;
    const size_t N = o->N;
    double *ht = o->H2;      /* streamed populations */
    double *phin = o->C2;

    /* P1: stream-pull with periodic wrap / half-way bounce-back (A13, A16) */
#pragma omp parallel for collapse(2) schedule(static)
    for (int z = 0; z < o->nz; ++z)
        for (int y = 0; y < o->ny; ++y)
            for (int x = 0; x < o->nx; ++x) {
                size_t c = cell(o, x, y, z), nb;
                for (int i = 0; i < Q; ++i) {
                    if (neighbour(o, x, y, z, L->e[i], -1, &nb)) ht[i * N + c] = o->H[L->opp[i] * N + c];
                    else ht[i * N + c] = o->H[i * N + nb];
                }
            }
    /* P2: phi_new = sum_i h_i, eq. 7 */
#pragma omp parallel for schedule(static)
    for (size_t c = 0; c < N; ++c) {
        double s = 0.0;
        for (int i = 0; i < Q; ++i) s += ht[i * N + c];
        phin[c] = s;
    }
    /* P3 + P4: forcing (eq. 5) from the PREVIOUS phi field (A11), collision eq. 4 */
#pragma omp parallel for collapse(2) schedule(static)
    for (int z = 0; z < o->nz; ++z)
        for (int y = 0; y < o->ny; ++y)
            for (int x = 0; x < o->nx; ++x) {
                size_t c = cell(o, x, y, z);
                double g[3], n[3], F[QMAX], heq[QMAX], d[QMAX], m[QMAX], r[QMAX];
                grad_phi(o, L, o->C, x, y, z, g);
                double nrm = sqrt(g[0] * g[0] + g[1] * g[1] + g[2] * g[2]);
                for (int a = 0; a < 3; ++a) n[a] = (nrm > 0.0) ? g[a] / nrm : 0.0;
                double dphi = o->C[c] - PHI_0;
                double theta = (1.0 - 4.0 * dphi * dphi) / o->xi;               /* A1 */
                double u[3] = {o->U[c], o->U[N + c], o->U[2 * N + c]};
                for (int i = 0; i < Q; ++i) {
                    double en = L->e[i][0] * n[0] + L->e[i][1] * n[1] + L->e[i][2] * n[2];
                    F[i] = theta * L->w[i] * en;                                 /* eq. 5, dt = 1 */
                    heq[i] = phin[c] * Gamma(L, i, u);
                    d[i] = heq[i] - ht[i * N + c] - 0.5 * F[i];
                }
                /* Omega d = M^-1 S M d ; S: first-order moments omega_phi, others 1 (A2, A3);
                 * SRT variant (A23): every moment relaxes with omega_phi */
                const int srt = (o->variant & ORACLE_VAR_PHASE_SRT) != 0;
                matvec(Q, L->M, d, m);
                for (int k = 0; k < Q; ++k) m[k] *= (srt || L->order[k] == 1) ? o->omega_phi : 1.0;
                matvec(Q, L->Minv, m, r);
                for (int i = 0; i < Q; ++i) o->tmp[i * N + c] = r[i] + ht[i * N + c] + F[i];   /* eq. 4 */
            }
    /* P5: swap */
    memcpy(o->H, o->tmp, sizeof(double) * Q * N);
    memcpy(o->C, phin, sizeof(double) * N);
}

/* ------------------------------------------------------------------------- */
/* Hydrodynamic LB step (Alg. 2 lines 7-10): collide, stream-push, u    */
/* ------------------------------------------------------------------------- */

static void hydro_step(oracle_ctx *o)
{
    const lattice_t *L = &o->Lg;
    const int Q = L->Q;
    const size_t N = o->N;
    double *gs = o->tmp;     /* post-collision populations */

#pragma omp parallel for collapse(2) schedule(static)
    for (int z = 0; z < o->nz; ++z)
        for (int y = 0; y < o->ny; ++y)
            for (int x = 0; x < o->nx; ++x) {
                size_t c = cell(o, x, y, z);
                double g[QMAX];
                for (int i = 0; i < Q; ++i) g[i] = o->G[i * N + c];
                /* H1 */
                double pstar = 0.0;                                              /* eq. 15 */
                for (int i = 0; i < Q; ++i) pstar += g[i];
                double phi = o->C[c];                                            /* NEW phi (A12) */
                double rho = o->rho_L + (phi - PHI_L) * (o->rho_H - o->rho_L);   /* eq. 8 */
                double gphi[3], grho[3];
                grad_phi(o, L, o->C, x, y, z, gphi);
                double lap = lap_phi(o, L, o->C, x, y, z);
                double mu = 4.0 * o->beta * (phi - PHI_L) * (phi - PHI_H) * (phi - PHI_0) - o->kappa * lap; /* eq. 17 */
                for (int a = 0; a < 3; ++a) grho[a] = (o->rho_H - o->rho_L) * gphi[a];       /* A15 */
                double tau = o->tau_L + (phi - PHI_L) * (o->tau_H - o->tau_L);   /* eq. 20 */
                double s_nu = 1.0 / (tau + 0.5);                                 /* eq. 21 */
                double S[QMAX];
                /* A4: the six second-order moments relax with s_nu, all others with 1.  Variant A26: the
                 * lattice was built with the bulk moment as a row of its own (order ORDER_BULK), which then
                 * falls under "all others". */
                for (int k = 0; k < Q; ++k) S[k] = (L->order[k] == 2) ? s_nu : 1.0;

                /* H2: viscous force eq. 18 (A9) with u of the previous step (A10); variant A27 repeats
                 * H2 + H3 with the velocity just obtained (fixed point of eq. 22), o->subiter sweeps */
                double uo[3] = {o->U[c], o->U[N + c], o->U[2 * N + c]};
                double neq[QMAX], m[QMAX], v[QMAX];
                double F[3], un[3];
                for (int sweep = 0; sweep < o->subiter; ++sweep) {
                    for (int i = 0; i < Q; ++i) neq[i] = g[i] - (pstar * L->w[i] + Gamma(L, i, uo) - L->w[i]);  /* eq. 12 */
                    matvec(Q, L->M, neq, m);
                    for (int k = 0; k < Q; ++k) m[k] *= S[k];
                    matvec(Q, L->Minv, m, v);                                        /* Omega (g - geq) */
                    double nu = tau * CS2;                                           /* eq. 19 */
                    double Fmu[3];
                    for (int a = 0; a < 3; ++a) {
                        double acc = 0.0;
                        for (int b = 0; b < 3; ++b) {
                            double Pi = 0.0;
                            for (int k = 0; k < Q; ++k) Pi += L->e[k][a] * L->e[k][b] * v[k];
                            acc += Pi * grho[b];
                        }
                        Fmu[a] = -(nu / CS2) * acc;
                    }
                    for (int a = 0; a < 3; ++a)
                        F[a] = mu * gphi[a]                       /* F_s, eq. 16 */
                             - pstar * CS2 * grho[a]              /* F_p, eq. 14 */
                             + Fmu[a]                             /* F_mu, eq. 18 */
                             + rho * o->grav[a];                  /* F_b, eq. 30 (A17) */
                    /* H3: velocity, eq. 22 */
                    for (int a = 0; a < 3; ++a) {
                        double j = 0.0;
                        for (int i = 0; i < Q; ++i) j += g[i] * L->e[i][a];
                        un[a] = j + F[a] / (2.0 * rho);
                    }
                    for (int a = 0; a < 3; ++a) uo[a] = un[a];
                }
                /* H4: collision in moment space, eq. 25 as in the listing P:229 (A6) */
                double geq[QMAX], Fi[QMAX], meq[QMAX], Fm[QMAX], out[QMAX];
                for (int i = 0; i < Q; ++i) {
                    geq[i] = pstar * L->w[i] + Gamma(L, i, un) - L->w[i];        /* eq. 12 */
                    double eF = L->e[i][0] * F[0] + L->e[i][1] * F[1] + L->e[i][2] * F[2];
                    Fi[i] = L->w[i] * eF / (rho * CS2);                          /* eq. 11 */
                }
                matvec(Q, L->M, g, m);
                matvec(Q, L->M, geq, meq);
                matvec(Q, L->M, Fi, Fm);
                for (int k = 0; k < Q; ++k) m[k] = m[k] - (m[k] - meq[k] + 0.5 * Fm[k]) * S[k] + Fm[k];
                matvec(Q, L->Minv, m, out);
                for (int i = 0; i < Q; ++i) gs[i * N + c] = out[i];
                for (int a = 0; a < 3; ++a) o->U2[a * N + c] = un[a];
            }
    /* H5: stream-push with periodic wrap / half-way bounce-back (A13, A16) */
#pragma omp parallel for collapse(2) schedule(static)
    for (int z = 0; z < o->nz; ++z)
        for (int y = 0; y < o->ny; ++y)
            for (int x = 0; x < o->nx; ++x) {
                size_t c = cell(o, x, y, z), nb;
                for (int i = 0; i < Q; ++i) {
                    if (neighbour(o, x, y, z, L->e[i], +1, &nb)) o->G2[L->opp[i] * N + c] = gs[i * N + c];
                    else o->G2[i * N + nb] = gs[i * N + c];
                }
            }
    /* H6: swap */
    memcpy(o->G, o->G2, sizeof(double) * Q * N);
    memcpy(o->U, o->U2, sizeof(double) * 3 * N);
}

/* ------------------------------------------------------------------------- */
/* C interface (host pointers throughout)                                      */
/* ------------------------------------------------------------------------- */

int oracle_create(oracle_ctx **out, int nx, int ny, int nz, int stencil_phase, int stencil_hydro,
                  double rho_H, double rho_L, double sigma, double xi, double Mob, double nu_H, double nu_L,
                  const double gravity[3], unsigned wall_flags)
{
    if (!out) return 1;
    *out = NULL;
    if (nx <= 0 || ny <= 0 || nz <= 0 || rho_L <= 0 || rho_H < rho_L || xi <= 0 || Mob <= 0 || nu_H <= 0 || nu_L <= 0)
        return 1;
    oracle_ctx *o = (oracle_ctx *)calloc(1, sizeof(oracle_ctx));
    if (!o) return 3;
    o->nx = nx; o->ny = ny; o->nz = nz; o->N = (size_t)nx * ny * nz;
    if (build_lattice(stencil_phase, &o->Lh, 0) || build_lattice(stencil_hydro, &o->Lg, 0)) { free(o); return 1; }
    o->subiter = 1;
    /* two-dimensional instance: both lattices D2Q9, one plane, no z component of gravity */
    if ((stencil_phase == 9) != (stencil_hydro == 9)) { free(o); return 1; }
    if (stencil_phase == 9 && (nz != 1 || (gravity && gravity[2] != 0.0))) { free(o); return 1; }
    o->rho_H = rho_H; o->rho_L = rho_L; o->sigma = sigma; o->xi = xi; o->Mob = Mob; o->nu_H = nu_H; o->nu_L = nu_L;
    for (int a = 0; a < 3; ++a) o->grav[a] = gravity ? gravity[a] : 0.0;
    o->walls = wall_flags;
    double tau_phi = Mob / CS2;                /* eq. 2, dt = 1 */
    o->omega_phi = 1.0 / (tau_phi + 0.5);      /* A2 */
    o->beta = 12.0 * sigma / xi;
    o->kappa = 3.0 * sigma * xi / 2.0;
    o->tau_H = nu_H / CS2;                     /* eq. 19 */
    o->tau_L = nu_L / CS2;
    const size_t N = o->N;
    const int Qh = o->Lh.Q, Qg = o->Lg.Q, Qm = Qh > Qg ? Qh : Qg;
    o->H = (double *)calloc(Qh * N, sizeof(double)); o->H2 = (double *)calloc(Qh * N, sizeof(double));
    o->G = (double *)calloc(Qg * N, sizeof(double)); o->G2 = (double *)calloc(Qg * N, sizeof(double));
    o->C = (double *)calloc(N, sizeof(double)); o->C2 = (double *)calloc(N, sizeof(double));
    o->U = (double *)calloc(3 * N, sizeof(double)); o->U2 = (double *)calloc(3 * N, sizeof(double));
    o->tmp = (double *)calloc(Qm * N, sizeof(double));
    if (!o->H || !o->H2 || !o->G || !o->G2 || !o->C || !o->C2 || !o->U || !o->U2 || !o->tmp) return 3;
    *out = o;
    return 0;
}

void oracle_destroy(oracle_ctx *o)
{
    if (!o) return;
    free(o->H); free(o->H2); free(o->G); free(o->G2); free(o->C); free(o->C2); free(o->U); free(o->U2); free(o->tmp);
    free(o);
}

/* equilibrium initialiser (A14): C = phi, U = u, h_i = phi Gamma_i(u), g_i = Gamma_i(u) - w_i */
int oracle_init(oracle_ctx *o, const double *phi, const double *u)
{
    if (!o || !phi || !u) return 1;
    const size_t N = o->N;
    memcpy(o->C, phi, sizeof(double) * N);
    memcpy(o->U, u, sizeof(double) * 3 * N);
    for (size_t c = 0; c < N; ++c) {
        double uc[3] = {u[c], u[N + c], u[2 * N + c]};
        for (int i = 0; i < o->Lh.Q; ++i) o->H[i * N + c] = phi[c] * Gamma(&o->Lh, i, uc);
        for (int i = 0; i < o->Lg.Q; ++i) o->G[i * N + c] = Gamma(&o->Lg, i, uc) - o->Lg.w[i];
    }
    o->initialised = 1;
    return 0;
}

int oracle_step(oracle_ctx *o, int n)
{
    if (!o || n < 0) return 1;
    if (!o->initialised) return 2;
    for (int t = 0; t < n; ++t) {
        phase_step(o);     /* A12 */
        hydro_step(o);
    }
    return 0;
}

int oracle_fields(oracle_ctx *o, double *phi, double *u, double *p)
{
    if (!o) return 1;
    const size_t N = o->N;
    if (phi) memcpy(phi, o->C, sizeof(double) * N);
    if (u) memcpy(u, o->U, sizeof(double) * 3 * N);
    if (p)
        for (size_t c = 0; c < N; ++c) {
            double pstar = 0.0;
            for (int i = 0; i < o->Lg.Q; ++i) pstar += o->G[i * N + c];
            double rho = o->rho_L + (o->C[c] - PHI_L) * (o->rho_H - o->rho_L);
            p[c] = pstar * rho * CS2;                                           /* P:118, A19 */
        }
    return 0;
}

/* sum_x phi(x), Neumaier-compensated */
int oracle_phi_mass(oracle_ctx *o, double *total)
{
    if (!o || !total) return 1;
    double s = 0.0, comp = 0.0;
    for (size_t c = 0; c < o->N; ++c) {
        double v = o->C[c], t = s + v;
        comp += (fabs(s) >= fabs(v)) ? (s - t) + v : (v - t) + s;
        s = t;
    }
    *total = s + comp;
    return isfinite(*total) ? 0 : 4;
}

int oracle_get_pdfs(oracle_ctx *o, double *h, double *g)
{
    if (!o) return 1;
    if (h) memcpy(h, o->H, sizeof(double) * o->Lh.Q * o->N);
    if (g) memcpy(g, o->G, sizeof(double) * o->Lg.Q * o->N);
    return 0;
}

/* test access to the state (lets a test plant arbitrary PDFs) */
int oracle_set_pdfs(oracle_ctx *o, const double *h, const double *g)
{
    if (!o) return 1;
    if (h) memcpy(o->H, h, sizeof(double) * o->Lh.Q * o->N);
    if (g) memcpy(o->G, g, sizeof(double) * o->Lg.Q * o->N);
    return 0;
}

/* table access for the pin tests */
int oracle_lattice(int Q, int *e /*Q*3*/, double *w /*Q*/, int *opp, double *M /*Q*Q*/, double *Minv, int *order)
{
    lattice_t L;
    const int bulk_split = Q < 0;      /* -Q: the basis of variant A26 (bulk row has order ORDER_BULK) */
    if (bulk_split) Q = -Q;
    if (build_lattice(Q, &L, bulk_split)) return 1;
    for (int i = 0; i < Q; ++i) {
        if (e) { e[3 * i] = L.e[i][0]; e[3 * i + 1] = L.e[i][1]; e[3 * i + 2] = L.e[i][2]; }
        if (w) w[i] = L.w[i];
        if (opp) opp[i] = L.opp[i];
        if (order) order[i] = L.order[i];
    }
    if (M) memcpy(M, L.M, sizeof(double) * Q * Q);
    if (Minv) memcpy(Minv, L.Minv, sizeof(double) * Q * Q);
    return 0;
}

/* FD operators on a caller-supplied field (pin: exact on polynomials) */
int oracle_fd(oracle_ctx *o, int use_hydro_stencil, const double *C, double *grad /*3N*/, double *lap /*N*/)
{
    if (!o || !C) return 1;
    const lattice_t *L = use_hydro_stencil ? &o->Lg : &o->Lh;
    const size_t N = o->N;
    for (int z = 0; z < o->nz; ++z)
        for (int y = 0; y < o->ny; ++y)
            for (int x = 0; x < o->nx; ++x) {
                size_t c = cell(o, x, y, z);
                double g[3];
                grad_phi(o, L, C, x, y, z, g);
                if (grad) { grad[c] = g[0]; grad[N + c] = g[1]; grad[2 * N + c] = g[2]; }
                if (lap) lap[c] = lap_phi(o, L, C, x, y, z);
            }
    return 0;
}

int oracle_set_variant(oracle_ctx *o, unsigned flags)
{
    if (!o || (flags & ~(unsigned)(ORACLE_VAR_PHASE_SRT | ORACLE_VAR_BULK_ONE))) return 1;
    if ((flags ^ o->variant) & ORACLE_VAR_BULK_ONE)      /* the hydrodynamic moment basis with / without the bulk row */
        if (build_lattice(o->Lg.Q, &o->Lg, (flags & ORACLE_VAR_BULK_ONE) != 0)) return 1;
    o->variant = flags;
    return 0;
}

/* variant A27: number of sweeps of the fixed point of eq. 22 (1 = the default reading A10) */
int oracle_set_subiter(oracle_ctx *o, int sweeps)
{
    if (!o || sweeps < 1 || sweeps > 64) return 1;
    o->subiter = sweeps;
    return 0;
}

/* Rising-bubble diagnostics (section 6.1).  The paper uses "the terminal velocity of the
 * bubbles" u_t in eq. 34 without saying how it is measured; reading A24: the cells of
 * the bubble are those with phi < phi_0 = 1/2, weighted with (phi_H - phi), i.e. with w = (1 - phi) [phi < 1/2]
 *   V = sum_x w,  X_b = sum_x w x_c / V,  u_b = sum_x w u / V,
 * x_c = cell centre (i + 1/2), plain coordinates (no periodic unwrapping).  (Without the restriction to
 * phi < 1/2 the sums pick up the 1e-4 compression of the heavy liquid over millions of cells.)
 * out = { V, X_b[3], u_b[3] }. */
int oracle_bubble_diag(oracle_ctx *o, double out[7])
{
    if (!o || !out) return 1;
    const size_t N = o->N;
    double V = 0.0, X[3] = {0, 0, 0}, Ub[3] = {0, 0, 0};
    for (int z = 0; z < o->nz; ++z)
        for (int y = 0; y < o->ny; ++y)
            for (int x = 0; x < o->nx; ++x) {
                size_t c = cell(o, x, y, z);
                double wgt = (o->C[c] < PHI_0) ? PHI_H - o->C[c] : 0.0;
                V += wgt;
                X[0] += wgt * (x + 0.5); X[1] += wgt * (y + 0.5); X[2] += wgt * (z + 0.5);
                for (int a = 0; a < 3; ++a) Ub[a] += wgt * o->U[a * N + c];
            }
    out[0] = V;
    for (int a = 0; a < 3; ++a) { out[1 + a] = X[a] / V; out[4 + a] = Ub[a] / V; }
    return 0;
}

/* Dimensionless groups of section 6.1 solved for the lattice parameters:
 *   t_ref = sqrt(D/g_y)                 (eq. 33)  =>  g_y   = D / t_ref^2
 *   Eo    = g_y rho_H D^2 / sigma       (eq. 32)  =>  sigma = g_y rho_H D^2 / Eo
 *   Re_Gr = rho_H sqrt(g_y D^3) / mu_H  (eq. 31)  =>  mu_H  = rho_H sqrt(g_y D^3) / Re_Gr
 *   rho* = rho_H/rho_L, mu* = mu_H/mu_L, nu = mu/rho
 * out = { g_y, sigma, nu_H, nu_L, rho_L }. */
int oracle_bubble_params(double Re_Gr, double Eo, double D, double t_ref, double rho_H, double rho_star,
                         double mu_star, double out[5])
{
    if (!out || !(Re_Gr > 0) || !(Eo > 0) || !(D > 0) || !(t_ref > 0) || !(rho_H > 0) || !(rho_star > 0) || !(mu_star > 0))
        return 1;
    double gy = D / (t_ref * t_ref);
    double sigma = gy * rho_H * D * D / Eo;
    double mu_H = rho_H * sqrt(gy * D * D * D) / Re_Gr;
    double rho_L = rho_H / rho_star;
    double mu_L = mu_H / mu_star;
    out[0] = gy; out[1] = sigma; out[2] = mu_H / rho_H; out[3] = mu_L / rho_L; out[4] = rho_L;
    return 0;
}

/* eq. 34: C_D^LBM = 4/3 g_y (rho_H - rho_L) D / (rho_H u_t^2) */
double oracle_drag_lbm(double gy, double rho_H, double rho_L, double D, double u_t)
{
    return (4.0 / 3.0) * gy * (rho_H - rho_L) * D / (rho_H * u_t * u_t);
}

/* eq. 35: C_D^exp = [ 2.67^(9/10) + (16/Re_Gr)^(9/10) ]^(10/9) */
double oracle_drag_exp(double Re_Gr)
{
    return pow(pow(2.67, 0.9) + pow(16.0 / Re_Gr, 0.9), 10.0 / 9.0);
}

int oracle_set_threads(int n)
{
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
    return omp_get_max_threads();
#else
    (void)n;
    return 1;
#endif
}
