/*
 * oracle/tcpo.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, fp64 CPU oracle of the coupled per-cell time step of the thermocapillary
 * central-moment phase-field lattice Boltzmann model of arxiv 2401.03041.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may
 * load this library.  It shares no source, header, table or helper with the CUDA path
 * (paper_2401_03041_b200/csrc, include/tcp.h); it even declares its own copy of the
 * parameter struct.  It is written to be checked against the paper by eye:
 *
 *   - every collision builds the dense Q x Q central-moment matrix K(u)_{m,i} = b_m(c_i - u)
 *     and solves K y = r by Gaussian elimination (the paper names the
 *     central-moment collision at PAPER.md:36, 182, 262 but prints no formula);
 *   - the time loop is Algorithm 1 / Algorithm 2: update h, then g, then
 *     f or the Runge-Kutta stages; two-grid pull streaming;
 *   - no blocking, no fusion, no algebraic shortcuts.
 *
 * Parity pins (tests/test_oracle_*.py): lattice weights (App. B), sum(phi) conservation,
 * tanh profile width, mobility decay, 1-D heat closed form, two-wall conduction, Poiseuille,
 * Laplace law, BGK reduction, layered-channel closed form (App. A), variant agreement,
 * Marangoni direction, FD operators exact on quadratics, reading S16 (tests/test_oracle_s16_rhocp.py), the
 * 1/(rho c_p) of eq. 4, the wetting ghost rule S20 (tests/test_oracle_wetting.py: wall-normal gradient of the inclined
 * tanh profile, sessile-droplet cap angle).
 * PARITY UNPINNED (the oracle *is* the definition): transients, the rates of
 * central moments of order >= 3 and of the trace, the lag choices S4/S10, corner ghosts on
 * domains with walls on more than one axis.
 *
 * Readings of the paper taken here are the S/G/A items of SURVEY.md 8(c), listed in DESIGN.md.
 */
#define _USE_MATH_DEFINES
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#ifndef M_PI
#define M_PI 3.14159265358979323846
#endif
#define QMAX 27
#define CS2 (1.0 / 3.0) /* lattice speed of sound squared, PAPER.md:82-86 (c_s^2), App. B */

enum { TCPO_OK = 0, TCPO_EINVAL = -1, TCPO_ENOMEM = -2, TCPO_EUNSUPPORTED = -4, TCPO_ESTATE = -5 };
enum { TCPO_LB_D3Q7 = 0, TCPO_LB_D3Q15, TCPO_LB_D3Q19, TCPO_LB_D3Q27, TCPO_RK2, TCPO_RK4 };
enum { TCPO_PERIODIC = 0, TCPO_WALLS = 1 };

/* The oracle's own declaration of the problem statement (same field order as the GPU library's
 * struct so the harness can fill both from one dict; deliberately not a shared header). */
typedef struct tcpo_params {
    unsigned struct_size;
    int precision, thermal, streaming; /* precision/streaming ignored: the oracle is fp64, two-grid */
    int bc[3];
    double rho_H, rho_L;               /* eq. 14 */
    double tau_H, tau_L;               /* eq. 22; nu = tau c_s^2 */
    double xi, M;                      /* eqs. 3, 11, 15 */
    double sigma_ref, sigma_T, T_ref;  /* eq. 9 */
    double kappa_H, kappa_L, cp_H, cp_L; /* eqs. 23-24 PAPER.md:138-140 (reading G5) */
    double gravity[3];                 /* eq. 7 */
    double wall_T[3][2];
    double s_bulk, s_high;             /* reading S2 */
    int high_rate_equals_shear;        /* 1 => every rate = the physical one => BGK */
    double eps_normal;                 /* reading S8 */
    double wall_u[3][2][3];            /* wall velocity per axis / face (moving wall; reading S18) */
    double sigma_TT;                   /* d^2 sigma / dT^2: "parabolic (or non-linear) relation between surface tension and
                                          temperature" (reading S19); 0 = the linear eq. 9 */
    double wall_contact_angle[3][2];   /* contact angle theta in degrees of each wall [axis][face], measured inside the phi = 1 fluid
                                          (wetting boundary condition; reading S20); 90 = neutral = mirror ghost */
    int hydro_lattice;                 /* 27 (default) or 19: lattice of the hydrodynamic populations g ("hydrodynamic LBM solvers
                                          often rely on a D3Q19 or D3Q27 stencil"); weights App. B.3, basis S2 */
    int collision_space;               /* 0 (default): central moments, K(u)_{m,i} = b_m(c_i - u); 1: raw moments, K(0) -- the
                                          multiple-relaxation-time (MRT) operator with the same basis and rates ("the SRT or MRT methods
                                          retain widespread usage") */
    int equilibrium;                   /* 0 (default): the second-order equilibria printed in the paper (eqs. 12, 18); 1: the continuous
                                          Maxwellian taken in central-moment space (D3Q27 lattices only): central moments of x^a y^b z^c
                                          = s m_a m_b m_c with m_0 = 1, m_1 = 0, m_2 = c_s^2, in place of those of eq. 12; eq. 18
                                          becomes w_i (p* - 1) + that equilibrium with s = 1 */
    /* ---- oracle-only switches (no counterpart in the CUDA library) ---- */
    int hydro_phi_level;               /* which phi the hydrodynamic update differentiates: 0 = phi^n (reading S16, what
                                          Algorithm 1's communication order implies), 1 = phi^{n+1}
                                          (SURVEY O5's proposal).  Exists so that tests/test_oracle_s16.py can show what
                                          the alternative does on the paper's own channel benchmark */
} tcpo_params;

/* ------------------------------------------------------------------------------------------ */
/* lattices (App. B) and central-moment bases (reading S2)                   */

typedef struct {
    int Q;
    int c[QMAX][3];
    double w[QMAX];
    int opp[QMAX];
    /* basis function m = sum_{t<nterm[m]} x^e[m][t][0] y^e[m][t][1] z^e[m][t][2] */
    int nterm[QMAX];
    int e[QMAX][3][3];
    int order[QMAX];
    int ixx, iyy, izz; /* positions of x^2, y^2, z^2 in the basis */
} lattice;

static void add_basis(lattice *L, int *m, int nterm, const int e[][3]) {
    L->nterm[*m] = nterm;
    for (int t = 0; t < nterm; t++)
        for (int a = 0; a < 3; a++) L->e[*m][t][a] = e[t][a];
    L->order[*m] = e[0][0] + e[0][1] + e[0][2];
    if (nterm == 1 && e[0][0] == 2 && e[0][1] == 0 && e[0][2] == 0) L->ixx = *m;
    if (nterm == 1 && e[0][0] == 0 && e[0][1] == 2 && e[0][2] == 0) L->iyy = *m;
    if (nterm == 1 && e[0][0] == 0 && e[0][1] == 0 && e[0][2] == 2) L->izz = *m;
    (*m)++;
}

/* Q in {7,15,19,27}.  Velocity order: rest, 6 axis, 12 face diagonals, 8 corners (App. B
 * groups q=0 / 1..6 / 7..18 / 19..26), keeping only the groups the stencil has. */
static int lattice_build(lattice *L, int Q) {
    static const double W27[4] = {64.0 / 216, 16.0 / 216, 4.0 / 216, 1.0 / 216}; /* B.4 */
    static const double W19[4] = {12.0 / 36, 2.0 / 36, 1.0 / 36, 0.0};           /* B.3 */
    static const double W15[4] = {16.0 / 72, 8.0 / 72, 0.0, 1.0 / 72};           /* B.2 */
    static const double W7[4] = {0.0, 1.0 / 6, 0.0, 0.0};                        /* B.1 (w_0 = 0) */
    const double *W;
    int has[4] = {1, 1, 0, 0};
    memset(L, 0, sizeof *L);
    switch (Q) {
    case 27: W = W27; has[2] = has[3] = 1; break;
    case 19: W = W19; has[2] = 1; break;
    case 15: W = W15; has[3] = 1; break;
    case 7: W = W7; break;
    default: return -1;
    }
    int n = 0;
    for (int grp = 0; grp < 4; grp++) {
        if (!has[grp]) continue;
        for (int cz = -1; cz <= 1; cz++)
            for (int cy = -1; cy <= 1; cy++)
                for (int cx = -1; cx <= 1; cx++) {
                    if (abs(cx) + abs(cy) + abs(cz) != grp) continue;
                    L->c[n][0] = cx; L->c[n][1] = cy; L->c[n][2] = cz;
                    L->w[n] = W[grp];
                    n++;
                }
    }
    if (n != Q) return -1;
    L->Q = Q;
    for (int i = 0; i < Q; i++)
        for (int j = 0; j < Q; j++)
            if (L->c[j][0] == -L->c[i][0] && L->c[j][1] == -L->c[i][1] && L->c[j][2] == -L->c[i][2])
                L->opp[i] = j;
    /* basis (reading S2) */
    int m = 0;
    L->ixx = L->iyy = L->izz = -1;
    if (Q == 27 || Q == 19) {
        for (int ord = 0; ord <= 6; ord++)
            for (int a = 0; a <= 2; a++)
                for (int b = 0; b <= 2; b++)
                    for (int cc = 0; cc <= 2; cc++) {
                        if (a + b + cc != ord) continue;
                        if (Q == 19 && a * b * cc != 0) continue;
                        const int e[1][3] = {{a, b, cc}};
                        add_basis(L, &m, 1, e);
                    }
    } else if (Q == 7) {
        const int e[7][1][3] = {{{0, 0, 0}}, {{1, 0, 0}}, {{0, 1, 0}}, {{0, 0, 1}},
                                {{2, 0, 0}}, {{0, 2, 0}}, {{0, 0, 2}}};
        for (int k = 0; k < 7; k++) add_basis(L, &m, 1, e[k]);
    } else { /* Q == 15 */
        const int e1[11][1][3] = {{{0, 0, 0}}, {{1, 0, 0}}, {{0, 1, 0}}, {{0, 0, 1}},
                                  {{2, 0, 0}}, {{0, 2, 0}}, {{0, 0, 2}},
                                  {{1, 1, 0}}, {{1, 0, 1}}, {{0, 1, 1}}, {{1, 1, 1}}};
        for (int k = 0; k < 11; k++) add_basis(L, &m, 1, e1[k]);
        const int ex[2][3] = {{1, 2, 0}, {1, 0, 2}}; /* x (y^2 + z^2) */
        const int ey[2][3] = {{2, 1, 0}, {0, 1, 2}}; /* y (x^2 + z^2) */
        const int ez[2][3] = {{2, 0, 1}, {0, 2, 1}}; /* z (x^2 + y^2) */
        const int e4[3][3] = {{2, 2, 0}, {2, 0, 2}, {0, 2, 2}}; /* x^2y^2 + x^2z^2 + y^2z^2 */
        add_basis(L, &m, 2, ex);
        add_basis(L, &m, 2, ey);
        add_basis(L, &m, 2, ez);
        add_basis(L, &m, 3, e4);
    }
    if (m != Q) return -1;
    return 0;
}

static double ipow(double x, int n) { return n == 0 ? 1.0 : (n == 1 ? x : x * x); }

/* K(u)_{m,i} = b_m(c_i - u)   (generic collision operator) */
static void build_K(const lattice *L, const double u[3], double K[QMAX][QMAX]) {
    for (int m = 0; m < L->Q; m++)
        for (int i = 0; i < L->Q; i++) {
            double dx = L->c[i][0] - u[0], dy = L->c[i][1] - u[1], dz = L->c[i][2] - u[2];
            double s = 0.0;
            for (int t = 0; t < L->nterm[m]; t++)
                s += ipow(dx, L->e[m][t][0]) * ipow(dy, L->e[m][t][1]) * ipow(dz, L->e[m][t][2]);
            K[m][i] = s;
        }
}

/* Solve A y = b (n <= QMAX) by Gaussian elimination with partial pivoting; A, b destroyed. */
static int solve_dense(int n, double A[QMAX][QMAX], double *b, double *y) {
    for (int k = 0; k < n; k++) {
        int p = k;
        double best = fabs(A[k][k]);
        for (int r = k + 1; r < n; r++)
            if (fabs(A[r][k]) > best) { best = fabs(A[r][k]); p = r; }
        if (best == 0.0) return -1;
        if (p != k) {
            for (int cidx = 0; cidx < n; cidx++) { double t = A[k][cidx]; A[k][cidx] = A[p][cidx]; A[p][cidx] = t; }
            double t = b[k]; b[k] = b[p]; b[p] = t;
        }
        for (int r = k + 1; r < n; r++) {
            double f = A[r][k] / A[k][k];
            if (f == 0.0) continue;
            for (int cidx = k; cidx < n; cidx++) A[r][cidx] -= f * A[k][cidx];
            b[r] -= f * b[k];
        }
    }
    for (int k = n - 1; k >= 0; k--) {
        double s = b[k];
        for (int cidx = k + 1; cidx < n; cidx++) s -= A[k][cidx] * y[cidx];
        y[k] = s / A[k][k];
    }
    return 0;
}

/* relaxation rates of the central moments (reading S2) */
typedef struct {
    double r0, r1;      /* orders 0 and 1 */
    double r2s, r2b;    /* 2nd order: deviatoric (xy, xz, yz, and the two deviatoric diagonal combos) / trace */
    double r3;          /* order >= 3 */
} rates;

/* out = S in, in moment space.  For the diagonal 2nd-order moments:
 * (S D)_aa = r2s D_aa + (r2b - r2s) tr(D)/3. */
static void apply_S(const lattice *L, const rates *R, const double *in, double *out) {
    for (int m = 0; m < L->Q; m++) {
        switch (L->order[m]) {
        case 0: out[m] = R->r0 * in[m]; break;
        case 1: out[m] = R->r1 * in[m]; break;
        case 2: out[m] = R->r2s * in[m]; break;
        default: out[m] = R->r3 * in[m]; break;
        }
    }
    double tr = in[L->ixx] + in[L->iyy] + in[L->izz];
    out[L->ixx] = R->r2s * in[L->ixx] + (R->r2b - R->r2s) * tr / 3.0;
    out[L->iyy] = R->r2s * in[L->iyy] + (R->r2b - R->r2s) * tr / 3.0;
    out[L->izz] = R->r2s * in[L->izz] + (R->r2b - R->r2s) * tr / 3.0;
}

/* second-order equilibrium, eq. 12 for h (s = phi) and f (s = T):
 *   s w_i [1 + e_i.u/c_s^2 + (e_i.u)^2/(2 c_s^4) - u.u/(2 c_s^2)] */
static void eq_scalar(const lattice *L, double s, const double u[3], double *out) {
    double uu = u[0] * u[0] + u[1] * u[1] + u[2] * u[2];
    for (int i = 0; i < L->Q; i++) {
        double cu = L->c[i][0] * u[0] + L->c[i][1] * u[1] + L->c[i][2] * u[2];
        out[i] = s * L->w[i] * (1.0 + cu / CS2 + cu * cu / (2.0 * CS2 * CS2) - uu / (2.0 * CS2));
    }
}

/* incompressible equilibrium, eq. 18:
 *   w_i (p* + [e_i.u/c_s^2 + (e_i.u)^2/(2 c_s^4) - u.u/(2 c_s^2)]) */
static void eq_hydro(const lattice *L, double pstar, const double u[3], double *out) {
    double uu = u[0] * u[0] + u[1] * u[1] + u[2] * u[2];
    for (int i = 0; i < L->Q; i++) {
        double cu = L->c[i][0] * u[0] + L->c[i][1] * u[1] + L->c[i][2] * u[2];
        out[i] = L->w[i] * (pstar + (cu / CS2 + cu * cu / (2.0 * CS2 * CS2) - uu / (2.0 * CS2)));
    }
}

/* Maxwellian equilibrium in central-moment space (tcpo_params::equilibrium = 1), monomial bases only (D3Q27, D3Q19):
 * the populations a with K(u) a = kappa^M, kappa^M of x^a y^b z^c = s m_a m_b m_c, m = (1, 0, c_s^2) -- the central
 * moments of the continuous Maxwell-Boltzmann distribution of density s, velocity u, temperature c_s^2 on the basis. */
static int eq_scalar_maxwell(const lattice *L, double s, const double u[3], double *out) {
    static const double m1d[3] = {1.0, 0.0, CS2};
    double K[QMAX][QMAX], kap[QMAX];
    build_K(L, u, K);
    for (int m = 0; m < L->Q; m++) {
        if (L->nterm[m] != 1) return -1;
        kap[m] = s * m1d[L->e[m][0][0]] * m1d[L->e[m][0][1]] * m1d[L->e[m][0][2]];
    }
    return solve_dense(L->Q, K, kap, out);
}

/* eq. 18 with the bracket [...] = f_eq(rho = 1, u) / w_i - 1 taken from the Maxwellian: w_i (p* - 1) + a^M(1, u) */
static int eq_hydro_maxwell(const lattice *L, double pstar, const double u[3], double *out) {
    if (eq_scalar_maxwell(L, 1.0, u, out)) return -1;
    for (int i = 0; i < L->Q; i++) out[i] += L->w[i] * (pstar - 1.0);
    return 0;
}

/* Guo force populations (ref. [20] named at PAPER.md:100, 118):
 *   F_i(a,u) = w_i [ (c_i - u)/c_s^2 + (c_i.u) c_i / c_s^4 ] . a */
static void guo_populations(const lattice *L, const double a[3], const double u[3], double *out) {
    for (int i = 0; i < L->Q; i++) {
        double cu = L->c[i][0] * u[0] + L->c[i][1] * u[1] + L->c[i][2] * u[2];
        double s = 0.0;
        for (int al = 0; al < 3; al++)
            s += ((L->c[i][al] - u[al]) / CS2 + cu * L->c[i][al] / (CS2 * CS2)) * a[al];
        out[i] = L->w[i] * s;
    }
}

/* Generic central-moment collision:
 *   a~ = a - K^-1 S K (a - a_eq) + K^-1 (I - S/2) K F(avec, u)
 * computed as  r = S K (a - a_eq) - (K F - S K F / 2);  solve K y = r;  a~ = a - y. */
static int collide_generic(const lattice *L, const rates *R, const double u[3], const double *a,
                           const double *aeq, const double avec[3], double *out, int raw_space) {
    double K[QMAX][QMAX], d[QMAX], Fi[QMAX], kd[QMAX] = {0}, kf[QMAX] = {0}, skd[QMAX], skf[QMAX], r[QMAX], y[QMAX];
    int Q = L->Q;
    const double rest[3] = {0.0, 0.0, 0.0};
    build_K(L, raw_space ? rest : u, K); /* raw moments (MRT) = the same basis about the lattice at rest */
    guo_populations(L, avec, u, Fi);
    for (int i = 0; i < Q; i++) d[i] = a[i] - aeq[i];
    for (int m = 0; m < Q; m++) {
        double s1 = 0.0, s2 = 0.0;
        for (int i = 0; i < Q; i++) { s1 += K[m][i] * d[i]; s2 += K[m][i] * Fi[i]; }
        kd[m] = s1; kf[m] = s2;
    }
    apply_S(L, R, kd, skd);
    apply_S(L, R, kf, skf);
    for (int m = 0; m < Q; m++) r[m] = skd[m] - (kf[m] - 0.5 * skf[m]);
    if (solve_dense(Q, K, r, y) != 0) return -1;
    for (int i = 0; i < Q; i++) out[i] = a[i] - y[i];
    return 0;
}

/* ------------------------------------------------------------------------------------------ */
/* simulation state                                                                            */

typedef struct tcpo_sim {
    int nx, ny, nz;
    size_t N;
    tcpo_params P;
    lattice L27, LT, LH; /* D3Q27 for h and the FD stencils; LT for f; LH (D3Q27 or D3Q19) for g */
    int thermal_is_lb;
    double *h, *h2, *g, *g2, *f, *f2; /* post-collision populations [Q][N], two grids */
    double *phi, *phi2, *T, *T2, *u;  /* u = [3][N] */
    double *rk[4];                    /* RK work fields */
    double *wallT[3][2];              /* tangential-plane arrays */
    double *q;                        /* heat source or NULL */
    int initialised;
    long steps_done;
} tcpo_sim;

static __thread char g_err[256];
static int fail(int code, const char *msg) { snprintf(g_err, sizeof g_err, "%s", msg); return code; }
const char *tcpo_last_error(void) { return g_err; }

int tcpo_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* Threads for the cell loops of the calls that follow (the harness uses one thread on grids too small to
 * pay for a parallel region; the arithmetic per cell does not depend on it). */
void tcpo_set_num_threads(int n) {
#ifdef _OPENMP
    if (n >= 1) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

static size_t plane_size(const tcpo_sim *s, int axis) {
    return axis == 0 ? (size_t)s->ny * s->nz : (axis == 1 ? (size_t)s->nx * s->nz : (size_t)s->nx * s->ny);
}

int tcpo_destroy(tcpo_sim *s) {
    if (!s) return TCPO_OK;
    free(s->h); free(s->h2); free(s->g); free(s->g2); free(s->f); free(s->f2);
    free(s->phi); free(s->phi2); free(s->T); free(s->T2); free(s->u); free(s->q);
    for (int k = 0; k < 4; k++) free(s->rk[k]);
    for (int a = 0; a < 3; a++) for (int fc = 0; fc < 2; fc++) free(s->wallT[a][fc]);
    free(s);
    return TCPO_OK;
}

int tcpo_create(int nx, int ny, int nz, const tcpo_params *p, tcpo_sim **out) {
    if (!p || !out) return fail(TCPO_EINVAL, "null argument");
    if (p->struct_size != sizeof(tcpo_params)) return fail(TCPO_EINVAL, "struct_size mismatch");
    if (nx < 1 || ny < 1 || nz < 1) return fail(TCPO_EINVAL, "extent < 1");
    int n[3] = {nx, ny, nz};
    for (int a = 0; a < 3; a++) {
        if (p->bc[a] != TCPO_PERIODIC && p->bc[a] != TCPO_WALLS) return fail(TCPO_EINVAL, "bad bc");
        if (p->bc[a] == TCPO_WALLS && n[a] < 2) return fail(TCPO_EINVAL, "wall axis needs n >= 2");
    }
    if (p->thermal < TCPO_LB_D3Q7 || p->thermal > TCPO_RK4) return fail(TCPO_EINVAL, "bad thermal variant");
    if (p->hydro_lattice != 27 && p->hydro_lattice != 19) return fail(TCPO_EINVAL, "hydro_lattice must be 27 or 19");
    if (p->equilibrium != 0 && p->equilibrium != 1) return fail(TCPO_EINVAL, "equilibrium must be 0 (printed second-order) or 1 (Maxwellian)");
    if (p->equilibrium == 1 && (p->hydro_lattice != 27 || (p->thermal <= TCPO_LB_D3Q27 && p->thermal != TCPO_LB_D3Q27)))
        return fail(TCPO_EUNSUPPORTED, "Maxwellian equilibrium: D3Q27 lattices only (hydro_lattice = 27; thermal D3Q27 LB or RK)");
    if (p->collision_space != 0 && p->collision_space != 1) return fail(TCPO_EINVAL, "collision_space must be 0 (central) or 1 (raw)");
    if (!(p->tau_H > -0.5) || !(p->tau_L > -0.5)) return fail(TCPO_EINVAL, "tau <= -1/2");
    if (!(p->M > 0) || !(p->xi > 0)) return fail(TCPO_EINVAL, "M, xi must be > 0");
    if (!(p->rho_H > 0) || !(p->rho_L > 0)) return fail(TCPO_EINVAL, "rho must be > 0");
    if (!(p->kappa_H > 0) || !(p->kappa_L > 0) || !(p->cp_H > 0) || !(p->cp_L > 0))
        return fail(TCPO_EINVAL, "kappa, cp must be > 0");
    for (int a = 0; a < 3; a++)
        for (int fc = 0; fc < 2; fc++)
            if (!(p->wall_contact_angle[a][fc] >= 0.0 && p->wall_contact_angle[a][fc] <= 180.0))
                return fail(TCPO_EINVAL, "wall_contact_angle must lie in [0, 180] degrees");
    tcpo_sim *s = calloc(1, sizeof *s);
    if (!s) return fail(TCPO_ENOMEM, "calloc");
    s->nx = nx; s->ny = ny; s->nz = nz; s->N = (size_t)nx * ny * nz; s->P = *p;
    lattice_build(&s->L27, 27);
    lattice_build(&s->LH, p->hydro_lattice);
    static const int QT[4] = {7, 15, 19, 27};
    s->thermal_is_lb = p->thermal <= TCPO_LB_D3Q27;
    lattice_build(&s->LT, s->thermal_is_lb ? QT[p->thermal] : 7);
    size_t N = s->N;
    s->h = calloc(27 * N, 8); s->h2 = calloc(27 * N, 8);
    s->g = calloc((size_t)p->hydro_lattice * N, 8); s->g2 = calloc((size_t)p->hydro_lattice * N, 8);
    s->phi = calloc(N, 8); s->phi2 = calloc(N, 8);
    s->T = calloc(N, 8); s->T2 = calloc(N, 8); s->u = calloc(3 * N, 8);
    int ok = s->h && s->h2 && s->g && s->g2 && s->phi && s->phi2 && s->T && s->T2 && s->u;
    if (s->thermal_is_lb) {
        s->f = calloc((size_t)s->LT.Q * N, 8); s->f2 = calloc((size_t)s->LT.Q * N, 8);
        ok = ok && s->f && s->f2;
    } else {
        for (int k = 0; k < 4; k++) { s->rk[k] = calloc(N, 8); ok = ok && s->rk[k]; }
    }
    for (int a = 0; a < 3; a++)
        for (int fc = 0; fc < 2; fc++) {
            size_t m = plane_size(s, a);
            s->wallT[a][fc] = malloc(m * 8);
            if (!s->wallT[a][fc]) { ok = 0; continue; }
            for (size_t k = 0; k < m; k++) s->wallT[a][fc][k] = p->wall_T[a][fc];
        }
    if (!ok) { tcpo_destroy(s); return fail(TCPO_ENOMEM, "field allocation"); }
    *out = s;
    return TCPO_OK;
}

int tcpo_set_wall_temperature(tcpo_sim *s, int axis, int face, const double *Tw) {
    if (!s || axis < 0 || axis > 2 || face < 0 || face > 1) return fail(TCPO_EINVAL, "bad axis/face");
    size_t m = plane_size(s, axis);
    for (size_t k = 0; k < m; k++) s->wallT[axis][face][k] = Tw ? Tw[k] : s->P.wall_T[axis][face];
    return TCPO_OK;
}

int tcpo_set_heat_source(tcpo_sim *s, const double *q) {
    if (!s) return fail(TCPO_EINVAL, "null sim");
    free(s->q); s->q = NULL;
    if (q) {
        s->q = malloc(s->N * 8);
        if (!s->q) return fail(TCPO_ENOMEM, "q");
        memcpy(s->q, q, s->N * 8);
    }
    return TCPO_OK;
}

/* O0 ("initialising all fields"): h~ = h_eq(phi,u), g~ = g_eq(0,u), f~ = f_eq(T,u) */
int tcpo_init_fields(tcpo_sim *s, const double *phi, const double *u, const double *T) {
    if (!s || !phi) return fail(TCPO_EINVAL, "phi is required");
    size_t N = s->N;
    memcpy(s->phi, phi, N * 8);
    if (u) memcpy(s->u, u, 3 * N * 8); else memset(s->u, 0, 3 * N * 8);
    for (size_t k = 0; k < N; k++) s->T[k] = T ? T[k] : s->P.T_ref;
#pragma omp parallel for schedule(static)
    for (long k = 0; k < (long)N; k++) {
        double uu[3] = {s->u[k], s->u[N + k], s->u[2 * N + k]};
        double e[QMAX];
        const int mx = s->P.equilibrium == 1;
        if (mx) eq_scalar_maxwell(&s->L27, s->phi[k], uu, e); else eq_scalar(&s->L27, s->phi[k], uu, e);
        for (int i = 0; i < 27; i++) s->h[i * N + k] = e[i];
        if (mx) eq_hydro_maxwell(&s->LH, 0.0, uu, e); else eq_hydro(&s->LH, 0.0, uu, e);
        for (int i = 0; i < s->LH.Q; i++) s->g[i * N + k] = e[i];
        if (s->thermal_is_lb) {
            if (mx) eq_scalar_maxwell(&s->LT, s->T[k], uu, e); else
            eq_scalar(&s->LT, s->T[k], uu, e);
            for (int i = 0; i < s->LT.Q; i++) s->f[i * N + k] = e[i];
        }
    }
    s->initialised = 1;
    s->steps_done = 0;
    return TCPO_OK;
}

/* ------------------------------------------------------------------------------------------ */
/* neighbours, ghosts and pulls (reading S9)                                     */

/* coordinate i+d along an axis of extent n.  Periodic: wrapped, *face = -1.  Walls: if the
 * coordinate leaves the domain it is mirrored about the wall half a cell outside (-1 -> 0,
 * n -> n-1) and *face = 0 (low wall) or 1 (high wall). */
static int nb(int i, int d, int n, int bc, int *face) {
    int j = i + d;
    *face = -1;
    if (j < 0) { if (bc == TCPO_PERIODIC) j += n; else { *face = 0; j = 0; } }
    else if (j >= n) { if (bc == TCPO_PERIODIC) j -= n; else { *face = 1; j = n - 1; } }
    return j;
}

typedef struct { size_t idx; int axis, face; size_t tang; } nbr;

/* neighbour cell (x+dx, y+dy, z+dz).  axis = first wall axis crossed (x, then y, then z) or -1;
 * tang = index into that wall's tangential-plane array at the (wrapped / mirrored) tangential
 * coordinates of the requested cell. */
static nbr neighbour(const tcpo_sim *s, int x, int y, int z, int dx, int dy, int dz) {
    int fx, fy, fz;
    int X = nb(x, dx, s->nx, s->P.bc[0], &fx);
    int Y = nb(y, dy, s->ny, s->P.bc[1], &fy);
    int Z = nb(z, dz, s->nz, s->P.bc[2], &fz);
    nbr r;
    r.idx = (size_t)X + (size_t)s->nx * ((size_t)Y + (size_t)s->ny * Z);
    r.axis = -1; r.face = -1; r.tang = 0;
    if (fx >= 0) { r.axis = 0; r.face = fx; r.tang = (size_t)Z * s->ny + Y; }
    else if (fy >= 0) { r.axis = 1; r.face = fy; r.tang = (size_t)Z * s->nx + X; }
    else if (fz >= 0) { r.axis = 2; r.face = fz; r.tang = (size_t)Y * s->nx + X; }
    return r;
}

/* Wetting boundary condition (PAPER.md:307 names it -- "based on that proposed by Fakhari et al. [34]" -- and prints no
 * formula; reading S20).  At a wall with unit normal n_w pointing into the fluid the equilibrium profile
 * phi = 1/2 [1 + tanh(2 s / xi)] (eq. 35) that meets the wall at the contact angle theta (measured inside the
 * phi = 1 fluid) satisfies
 *     n_w . grad phi = Theta phi_w (1 - phi_w),      Theta = -(4 / xi) cos(theta)
 * (|grad phi| = (4/xi) phi (1 - phi) on that profile, and the interface normal grad phi / |grad phi| makes the angle
 * pi - theta with n_w).  With the wall half a cell outside the first fluid cell (S9): phi_w = (phi_f + phi_g) / 2 and
 * n_w . grad phi = (phi_f - phi_g) / 1, phi_f the fluid cell across the wall from the ghost cell.  Eliminating phi_g:
 *     a phi_w^2 - (1 + a) phi_w + phi_f = 0,   a = Theta / 2,
 * of which the root that tends to phi_f for a -> 0 is taken, and phi_g = 2 phi_w - phi_f.  theta = 90 degrees: a = 0,
 * phi_g = phi_f, the mirror ghost of S9.  The quadratic is solved the textbook cancellation-free way
 * (q = -(B + sgn(B) sqrt(B^2 - 4AC)) / 2, roots q / A and C / q; here B = -(1 + a) < 0 and the wanted root is C / q). */
static double wetting_ghost(const tcpo_sim *s, int axis, int face, double phi_f) {
    double theta = s->P.wall_contact_angle[axis][face];
    if (theta == 90.0) return phi_f;
    double a = 0.5 * (-(4.0 / s->P.xi) * cos(theta * M_PI / 180.0));
    double A = a, B = -(1.0 + a), C = phi_f;
    double q = -0.5 * (B - sqrt(B * B - 4.0 * A * C));
    double phi_w = C / q;
    return 2.0 * phi_w - phi_f;
}

/* phi at a neighbour: ghost from the mirror cell by the wetting condition (neutral wetting: the mirror cell's value) */
static double phi_at(const tcpo_sim *s, const double *phi, int x, int y, int z, int dx, int dy, int dz) {
    nbr r = neighbour(s, x, y, z, dx, dy, dz);
    if (r.axis >= 0) return wetting_ghost(s, r.axis, r.face, phi[r.idx]);
    return phi[r.idx];
}

/* a temperature-like field at a neighbour: ghost = 2 T_w - Y(mirror cell) */
static double temp_at(const tcpo_sim *s, const double *Y, int x, int y, int z, int dx, int dy, int dz) {
    nbr r = neighbour(s, x, y, z, dx, dy, dz);
    if (r.axis >= 0) return 2.0 * s->wallT[r.axis][r.face][r.tang] - Y[r.idx];
    return Y[r.idx];
}

/* Isotropic finite differences with the D3Q27 weights (reading S3):
 *   grad psi = (1/c_s^2) sum_i w_i c_i psi(x + c_i)
 *   lap  psi = (2/c_s^2) sum_i w_i [psi(x + c_i) - psi(x)]
 * is_temp selects the ghost rule. */
static void fd_ops(const tcpo_sim *s, const double *psi, int is_temp, int x, int y, int z, double grad[3], double *lap) {
    const lattice *L = &s->L27;
    double g0 = 0, g1 = 0, g2 = 0, l = 0;
    double centre = psi[(size_t)x + (size_t)s->nx * ((size_t)y + (size_t)s->ny * z)];
    for (int i = 0; i < 27; i++) {
        double v = is_temp ? temp_at(s, psi, x, y, z, L->c[i][0], L->c[i][1], L->c[i][2])
                           : phi_at(s, psi, x, y, z, L->c[i][0], L->c[i][1], L->c[i][2]);
        g0 += L->w[i] * L->c[i][0] * v;
        g1 += L->w[i] * L->c[i][1] * v;
        g2 += L->w[i] * L->c[i][2] * v;
        l += L->w[i] * (v - centre);
    }
    grad[0] = g0 / CS2; grad[1] = g1 / CS2; grad[2] = g2 / CS2;
    *lap = 2.0 * l / CS2;
}

/* pull(a~)_i(x) = a~_i(x - c_i); halfway bounce-back a~_ibar(x) if the link crosses a wall */
static double pull_bb(const tcpo_sim *s, const lattice *L, const double *a, int i, int x, int y, int z, size_t k) {
    nbr r = neighbour(s, x, y, z, -L->c[i][0], -L->c[i][1], -L->c[i][2]);
    if (r.axis >= 0) return a[(size_t)L->opp[i] * s->N + k];
    return a[(size_t)i * s->N + r.idx];
}

/* hydrodynamic pull: halfway bounce-back from a wall moving with U_w (reading S18):
 *   g_i(x) = g~_ibar(x) + 2 w_i (c_i . U_w) / c_s^2   (velocity-based model: no density factor);
 * h and f keep the plain (anti-)bounce-back of S9 */
static double pull_bb_moving(const tcpo_sim *s, const lattice *L, const double *a, int i, int x, int y, int z, size_t k) {
    nbr r = neighbour(s, x, y, z, -L->c[i][0], -L->c[i][1], -L->c[i][2]);
    if (r.axis >= 0) {
        const double *U = s->P.wall_u[r.axis][r.face];
        double cu = L->c[i][0] * U[0] + L->c[i][1] * U[1] + L->c[i][2] * U[2];
        return a[(size_t)L->opp[i] * s->N + k] + 2.0 * L->w[i] * cu / CS2;
    }
    return a[(size_t)i * s->N + r.idx];
}

/* thermal pull: Dirichlet wall by anti-bounce-back  -f~_ibar(x) + 2 w_i T_w */
static double pull_abb(const tcpo_sim *s, const lattice *L, const double *a, int i, int x, int y, int z, size_t k) {
    nbr r = neighbour(s, x, y, z, -L->c[i][0], -L->c[i][1], -L->c[i][2]);
    if (r.axis >= 0) return -a[(size_t)L->opp[i] * s->N + k] + 2.0 * L->w[i] * s->wallT[r.axis][r.face][r.tang];
    return a[(size_t)i * s->N + r.idx];
}

/* ------------------------------------------------------------------------------------------ */
/* the three updates of one time step                                                          */

static double lerp_phi(double lo, double hi, double phi) { return lo + phi * (hi - lo); } /* phi_L = 0 */

/* O1-O3: phase-field LB (eqs. 10-15) */
static int update_h(tcpo_sim *s) {
    const lattice *L = &s->L27;
    const tcpo_params *P = &s->P;
    size_t N = s->N;
    int bad = 0;
    double w_phi = 1.0 / (0.5 + P->M / CS2); /* eq. 11 read as a rate (G3) */
    rates R = {1.0, w_phi, 1.0, 1.0, 1.0};
    if (P->high_rate_equals_shear) { R.r0 = R.r1 = R.r2s = R.r2b = R.r3 = w_phi; }
#pragma omp parallel for collapse(2) schedule(static) reduction(| : bad)
    for (int z = 0; z < s->nz; z++)
        for (int y = 0; y < s->ny; y++)
            for (int x = 0; x < s->nx; x++) {
                size_t k = (size_t)x + (size_t)s->nx * ((size_t)y + (size_t)s->ny * z);
                double hp[QMAX], heq[QMAX], hout[QMAX];
                double phin = 0.0;
                for (int i = 0; i < 27; i++) { hp[i] = pull_bb(s, L, s->h, i, x, y, z, k); phin += hp[i]; } /* O1, eq. 13 */
                /* O2: interface force from the stored phi^n (S10), eq. 15 with the c_s^2 of S7 */
                double G[3], lap;
                fd_ops(s, s->phi, 0, x, y, z, G, &lap);
                double nrm = sqrt(G[0] * G[0] + G[1] * G[1] + G[2] * G[2] + P->eps_normal);
                double ph = s->phi[k];
                double mag = CS2 * (4.0 * ph * (1.0 - ph) / P->xi);
                double a[3] = {mag * G[0] / nrm, mag * G[1] / nrm, mag * G[2] / nrm};
                double u[3] = {s->u[k], s->u[N + k], s->u[2 * N + k]};
                if (P->equilibrium == 1) { if (eq_scalar_maxwell(L, phin, u, heq)) bad |= 1; }
                else eq_scalar(L, phin, u, heq); /* eq. 12 with phi' */
                if (collide_generic(L, &R, u, hp, heq, a, hout, P->collision_space)) bad |= 1;
                for (int i = 0; i < 27; i++) s->h2[(size_t)i * N + k] = hout[i];
                s->phi2[k] = phin;
            }
    if (bad) return fail(TCPO_ESTATE, "singular K in update_h");
    double *t = s->h; s->h = s->h2; s->h2 = t;
    /* phi^{n+1} stays in phi2 until update_g has run: the hydrodynamic update reads phi^n
     * (reading S16: Algorithm 1 exchanges phi once per step, after "update g",
     * PAPER.md:369-372, so the phi the g-update differentiates is the one from before this
     * step's h-update; with phi^{n+1} instead the coupled scheme pumps the staggered momentum
     * mode and the paper's own 4e5-step benchmark, would blow up). */
    return TCPO_OK;
}

/* O4-O7: hydrodynamic LB (eqs. 16-22 and 7-9) */
static int update_g(tcpo_sim *s) {
    const lattice *L = &s->LH;  /* D3Q27 or D3Q19 */
    const tcpo_params *P = &s->P;
    size_t N = s->N;
    int bad = 0;
    double drho = P->rho_H - P->rho_L;
#pragma omp parallel for collapse(2) schedule(static) reduction(| : bad)
    for (int z = 0; z < s->nz; z++)
        for (int y = 0; y < s->ny; y++)
            for (int x = 0; x < s->nx; x++) {
                size_t k = (size_t)x + (size_t)s->nx * ((size_t)y + (size_t)s->ny * z);
                double gp[QMAX], geq[QMAX], gout[QMAX];
                double pstar = 0.0, j[3] = {0, 0, 0};
                for (int i = 0; i < L->Q; i++) { /* O4, eq. 17 */
                    gp[i] = pull_bb_moving(s, L, s->g, i, x, y, z, k);
                    pstar += gp[i];
                    for (int al = 0; al < 3; al++) j[al] += L->c[i][al] * gp[i];
                }
                /* O5: local properties and finite differences of phi^n (S16), T^n */
                double ph = s->phi[k], Tc = s->T[k];
                double rho = lerp_phi(P->rho_L, P->rho_H, ph); /* eq. 14 */
                double tau = lerp_phi(P->tau_L, P->tau_H, ph); /* eq. 22 */
                double G[3], lap, Th[3], lapT;
                fd_ops(s, s->phi, 0, x, y, z, G, &lap);
                fd_ops(s, s->T, 1, x, y, z, Th, &lapT);
                /* eq. 9, plus the parabolic term of reading S19 (sigma_TT = 0: eq. 9 as printed);
                 * dsigma = d sigma / dT is what multiplies the tangential (Marangoni) term of eq. 8 */
                double dTr = Tc - P->T_ref;
                double sigma = P->sigma_ref + P->sigma_T * dTr + 0.5 * P->sigma_TT * dTr * dTr;
                double dsigma = P->sigma_T + P->sigma_TT * dTr;
                double beta = 12.0 * sigma / P->xi, kphi = 1.5 * sigma * P->xi; /* S5 */
                double mu = 4.0 * beta * ph * (ph - 1.0) * (ph - 0.5) - kphi * lap;
                /* O6: forces.  eq. 8 (with |grad phi|^2, G2), eq. 7, eq. 20 */
                double GG = G[0] * G[0] + G[1] * G[1] + G[2] * G[2];
                double TG = Th[0] * G[0] + Th[1] * G[1] + Th[2] * G[2];
                double F0[3], ustar[3], Fmu[3], F[3], u[3], a[3];
                for (int al = 0; al < 3; al++) {
                    double Fs = mu * G[al] + 1.5 * P->xi * dsigma * (GG * Th[al] - TG * G[al]);
                    double Fb = rho * P->gravity[al];
                    double Fp = -pstar * CS2 * drho * G[al];
                    F0[al] = Fs + Fb + Fp;
                    ustar[al] = j[al] + F0[al] / (2.0 * rho); /* predictor, S4 */
                }
                /* non-equilibrium second moments about g_eq(p*, u*) and eq. 21 */
                if (P->equilibrium == 1) { if (eq_hydro_maxwell(L, pstar, ustar, geq)) bad |= 1; }
                else eq_hydro(L, pstar, ustar, geq);
                double Pi[3][3] = {{0}};
                for (int i = 0; i < L->Q; i++)
                    for (int al = 0; al < 3; al++)
                        for (int be = 0; be < 3; be++) Pi[al][be] += L->c[i][al] * L->c[i][be] * (gp[i] - geq[i]);
                for (int al = 0; al < 3; al++) {
                    double t = 0.0;
                    for (int be = 0; be < 3; be++) t += Pi[al][be] * G[be];
                    Fmu[al] = -(tau / (tau + 0.5)) * drho * t;
                    F[al] = F0[al] + Fmu[al]; /* eq. 19 */
                    u[al] = j[al] + F[al] / (2.0 * rho); /* O7, S6 */
                    a[al] = F[al] / rho;
                }
                if (P->equilibrium == 1) { if (eq_hydro_maxwell(L, pstar, u, geq)) bad |= 1; }
                else eq_hydro(L, pstar, u, geq); /* eq. 18 */
                double om = 1.0 / (tau + 0.5);
                rates R = {1.0, 1.0, om, P->s_bulk, P->s_high};
                if (P->high_rate_equals_shear) { R.r0 = R.r1 = R.r2s = R.r2b = R.r3 = om; }
                if (collide_generic(L, &R, u, gp, geq, a, gout, P->collision_space)) bad |= 1;
                for (int i = 0; i < L->Q; i++) s->g2[(size_t)i * N + k] = gout[i];
                s->u[k] = u[0]; s->u[N + k] = u[1]; s->u[2 * N + k] = u[2]; /* u is only read locally */
            }
    if (bad) return fail(TCPO_ESTATE, "singular K in update_g");
    double *t = s->g; s->g = s->g2; s->g2 = t;
    return TCPO_OK;
}

/* O8-LB: thermal LB (eqs. 27-29); rho c_p = 1 on this path (S11) */
static int update_f(tcpo_sim *s) {
    const lattice *L = &s->LT;
    const tcpo_params *P = &s->P;
    size_t N = s->N;
    int bad = 0;
#pragma omp parallel for collapse(2) schedule(static) reduction(| : bad)
    for (int z = 0; z < s->nz; z++)
        for (int y = 0; y < s->ny; y++)
            for (int x = 0; x < s->nx; x++) {
                size_t k = (size_t)x + (size_t)s->nx * ((size_t)y + (size_t)s->ny * z);
                double fp[QMAX], feq[QMAX], fout[QMAX];
                double Tn = 0.0;
                for (int i = 0; i < L->Q; i++) { fp[i] = pull_abb(s, L, s->f, i, x, y, z, k); Tn += fp[i]; } /* eq. 28 */
                double kap = lerp_phi(P->kappa_L, P->kappa_H, s->phi[k]); /* eq. 23 (G5) */
                double w_T = 1.0 / (0.5 + kap / CS2);                      /* eq. 29 read as a rate (G4) */
                rates R = {1.0, w_T, 1.0, 1.0, 1.0};
                if (P->high_rate_equals_shear) { R.r0 = R.r1 = R.r2s = R.r2b = R.r3 = w_T; }
                double u[3] = {s->u[k], s->u[N + k], s->u[2 * N + k]};
                double zero[3] = {0, 0, 0};
                if (P->equilibrium == 1) { if (eq_scalar_maxwell(L, Tn, u, feq)) bad |= 1; }
                else eq_scalar(L, Tn, u, feq);
                if (collide_generic(L, &R, u, fp, feq, zero, fout, P->collision_space)) bad |= 1;
                double qT = s->q ? s->q[k] : 0.0;
                for (int i = 0; i < L->Q; i++) s->f2[(size_t)i * N + k] = fout[i] + L->w[i] * qT; /* eq. 27 */
                s->T2[k] = Tn;
            }
    if (bad) return fail(TCPO_ESTATE, "singular K in update_f");
    double *t = s->f; s->f = s->f2; s->f2 = t;
    t = s->T; s->T = s->T2; s->T2 = t;
    return TCPO_OK;
}

/* right-hand side of eq. 4 for a stage field Y, with phi^{n+1}, u^{n+1}:
 *   R(Y) = -u.grad Y + [grad kappa . grad Y + kappa lap Y] / (rho c_p) + q_T,
 *   grad kappa = (kappa_H - kappa_L) grad phi */
static void rk_rhs(const tcpo_sim *s, const double *Y, double *out) {
    const tcpo_params *P = &s->P;
    size_t N = s->N;
#pragma omp parallel for collapse(2) schedule(static)
    for (int z = 0; z < s->nz; z++)
        for (int y = 0; y < s->ny; y++)
            for (int x = 0; x < s->nx; x++) {
                size_t k = (size_t)x + (size_t)s->nx * ((size_t)y + (size_t)s->ny * z);
                double gY[3], lY, gP[3], lP;
                fd_ops(s, Y, 1, x, y, z, gY, &lY);
                fd_ops(s, s->phi, 0, x, y, z, gP, &lP);
                double ph = s->phi[k];
                double kap = lerp_phi(P->kappa_L, P->kappa_H, ph);
                double rcp = lerp_phi(P->rho_L, P->rho_H, ph) * lerp_phi(P->cp_L, P->cp_H, ph); /* A14 */
                double adv = s->u[k] * gY[0] + s->u[N + k] * gY[1] + s->u[2 * N + k] * gY[2];
                double dk = (P->kappa_H - P->kappa_L) * (gP[0] * gY[0] + gP[1] * gY[1] + gP[2] * gY[2]);
                out[k] = -adv + (dk + kap * lY) / rcp + (s->q ? s->q[k] : 0.0);
            }
}

/* O8-RK: eqs. 25-26, delta_t = 1 */
static int update_T_rk(tcpo_sim *s) {
    size_t N = s->N;
    double *K1 = s->rk[0], *K2 = s->rk[1], *K3 = s->rk[2], *Y = s->rk[3];
    if (s->P.thermal == TCPO_RK2) { /* eq. 26 with the T^n restored (G6) */
        rk_rhs(s, s->T, K1);
        for (size_t k = 0; k < N; k++) Y[k] = s->T[k] + 0.5 * K1[k];
        rk_rhs(s, Y, K2);
        for (size_t k = 0; k < N; k++) s->T[k] = s->T[k] + K2[k];
    } else { /* eq. 25 */
        double *K4 = s->T2;
        rk_rhs(s, s->T, K1);
        for (size_t k = 0; k < N; k++) Y[k] = s->T[k] + 0.5 * K1[k];
        rk_rhs(s, Y, K2);
        for (size_t k = 0; k < N; k++) Y[k] = s->T[k] + 0.5 * K2[k];
        rk_rhs(s, Y, K3);
        for (size_t k = 0; k < N; k++) Y[k] = s->T[k] + K3[k];
        rk_rhs(s, Y, K4);
        for (size_t k = 0; k < N; k++)
            s->T[k] = s->T[k] + K1[k] / 6.0 + K2[k] / 3.0 + K3[k] / 3.0 + K4[k] / 6.0;
    }
    return TCPO_OK;
}

/* Algorithm 1 / Algorithm 2: h, then g, then f or RK */
int tcpo_step(tcpo_sim *s, int nsteps) {
    if (!s) return fail(TCPO_EINVAL, "null sim");
    if (!s->initialised) return fail(TCPO_ESTATE, "tcpo_init_fields not called");
    if (nsteps < 0) return fail(TCPO_EINVAL, "nsteps < 0");
    for (int n = 0; n < nsteps; n++) {
        int rc;
        if ((rc = update_h(s))) return rc;
        if (s->P.hydro_phi_level == 1) { double *t = s->phi; s->phi = s->phi2; s->phi2 = t; } /* O5 as SURVEY proposed it */
        if ((rc = update_g(s))) return rc;
        if (s->P.hydro_phi_level != 1) { double *t = s->phi; s->phi = s->phi2; s->phi2 = t; } /* phi^{n+1} becomes current (S16) */
        if ((rc = s->thermal_is_lb ? update_f(s) : update_T_rk(s))) return rc;
        s->steps_done++;
    }
    return TCPO_OK;
}

/* Temperature pre-initialisation ("the temperature field is often times initialised by
 * executing the thermal solver until a certain error is reached"): the temperature update alone, with
 * phi, u, h~, g~ frozen. */
int tcpo_relax_temperature(tcpo_sim *s, int nsteps) {
    if (!s) return fail(TCPO_EINVAL, "null sim");
    if (!s->initialised) return fail(TCPO_ESTATE, "tcpo_init_fields not called");
    if (nsteps < 0) return fail(TCPO_EINVAL, "nsteps < 0");
    for (int n = 0; n < nsteps; n++) {
        int rc = s->thermal_is_lb ? update_f(s) : update_T_rk(s);
        if (rc) return rc;
    }
    return TCPO_OK;
}

/* O9: phi, u, T as stored; p = c_s^2 rho(phi) sum_i g~_i  (A12) */
int tcpo_read_fields(tcpo_sim *s, double *phi, double *u, double *p, double *T) {
    if (!s) return fail(TCPO_EINVAL, "null sim");
    if (!s->initialised) return fail(TCPO_ESTATE, "tcpo_init_fields not called");
    size_t N = s->N;
    if (phi) memcpy(phi, s->phi, N * 8);
    if (u) memcpy(u, s->u, 3 * N * 8);
    if (T) memcpy(T, s->T, N * 8);
    if (p)
        for (size_t k = 0; k < N; k++) {
            double ps = 0.0;
            for (int i = 0; i < s->LH.Q; i++) ps += s->g[(size_t)i * N + k];
            p[k] = CS2 * lerp_phi(s->P.rho_L, s->P.rho_H, s->phi[k]) * ps;
        }
    return TCPO_OK;
}

/* ------------------------------------------------------------------------------------------ */
/* small windows into the oracle for the pins                                                  */

/* populations: which = 0 (h), 1 (g), 2 (f); out = [Q][N] */
int tcpo_read_populations(tcpo_sim *s, int which, double *out) {
    if (!s || !out) return fail(TCPO_EINVAL, "null");
    const double *src = which == 0 ? s->h : (which == 1 ? s->g : s->f);
    int Q = which == 2 ? s->LT.Q : (which == 1 ? s->LH.Q : 27);
    if (!src) return fail(TCPO_ESTATE, "no such populations");
    memcpy(out, src, (size_t)Q * s->N * 8);
    return TCPO_OK;
}

/* lattice tables: c_out[Q][3], w_out[Q], opp_out[Q], order_out[Q] (order of basis function m) */
int tcpo_lattice(int Q, int *c_out, double *w_out, int *opp_out, int *order_out) {
    lattice L;
    if (lattice_build(&L, Q)) return fail(TCPO_EINVAL, "Q must be 7, 15, 19 or 27");
    for (int i = 0; i < Q; i++) {
        if (c_out) { c_out[3 * i] = L.c[i][0]; c_out[3 * i + 1] = L.c[i][1]; c_out[3 * i + 2] = L.c[i][2]; }
        if (w_out) w_out[i] = L.w[i];
        if (opp_out) opp_out[i] = L.opp[i];
        if (order_out) order_out[i] = L.order[i];
    }
    return TCPO_OK;
}

/* one generic collision on one cell.  kind: 0 scalar equilibrium (eq. 12) with moment s0,
 * 1 hydrodynamic equilibrium (eq. 18) with p* = s0.  rate5 = {r0, r1, r2s, r2b, r3}. */
int tcpo_collide_cell_space(int Q, int kind, const double *rate5, const double *u, double s0, const double *avec,
                            const double *a_in, double *a_out, int raw_space) {
    lattice L;
    if (lattice_build(&L, Q)) return fail(TCPO_EINVAL, "bad Q");
    rates R = {rate5[0], rate5[1], rate5[2], rate5[3], rate5[4]};
    double eq[QMAX];
    if (kind == 0) eq_scalar(&L, s0, u, eq); else eq_hydro(&L, s0, u, eq);
    if (collide_generic(&L, &R, u, a_in, eq, avec, a_out, raw_space)) return fail(TCPO_ESTATE, "singular K");
    return TCPO_OK;
}

int tcpo_collide_cell(int Q, int kind, const double *rate5, const double *u, double s0, const double *avec,
                      const double *a_in, double *a_out) {
    lattice L;
    if (lattice_build(&L, Q)) return fail(TCPO_EINVAL, "bad Q");
    rates R = {rate5[0], rate5[1], rate5[2], rate5[3], rate5[4]};
    double eq[QMAX];
    if (kind == 0) eq_scalar(&L, s0, u, eq); else eq_hydro(&L, s0, u, eq);
    if (collide_generic(&L, &R, u, a_in, eq, avec, a_out, 0)) return fail(TCPO_ESTATE, "singular K");
    return TCPO_OK;
}

/* central-moment matrix K(u) [Q][Q] row-major (row = basis function, column = velocity) */
int tcpo_central_moment_matrix(int Q, const double *u, double *K_out) {
    lattice L;
    double K[QMAX][QMAX];
    if (lattice_build(&L, Q)) return fail(TCPO_EINVAL, "bad Q");
    build_K(&L, u, K);
    for (int m = 0; m < Q; m++) for (int i = 0; i < Q; i++) K_out[m * Q + i] = K[m][i];
    return TCPO_OK;
}

/* grad and laplacian of a field with the sim's boundary rules; is_temp picks the ghost rule.
 * grad_out = [3][N], lap_out = [N] */
int tcpo_fd(tcpo_sim *s, const double *psi, int is_temp, double *grad_out, double *lap_out) {
    if (!s || !psi) return fail(TCPO_EINVAL, "null");
    size_t N = s->N;
    for (int z = 0; z < s->nz; z++)
        for (int y = 0; y < s->ny; y++)
            for (int x = 0; x < s->nx; x++) {
                size_t k = (size_t)x + (size_t)s->nx * ((size_t)y + (size_t)s->ny * z);
                double G[3], l;
                fd_ops(s, psi, is_temp, x, y, z, G, &l);
                if (grad_out) { grad_out[k] = G[0]; grad_out[N + k] = G[1]; grad_out[2 * N + k] = G[2]; }
                if (lap_out) lap_out[k] = l;
            }
    return TCPO_OK;
}
