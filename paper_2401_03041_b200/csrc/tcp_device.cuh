// Device-side building blocks of the coupled step: neighbourhoods and boundary rules, the
// isotropic finite differences, moments, and the closed-form central-moment collisions.
//
// Citations are PAPER.md:<line>.  Readings of the paper (S*/G*/A*) are listed in DESIGN.md.
// This file shares nothing with oracle/ (the CPU oracle builds dense moment matrices; here the
// same operator is evaluated in closed form).
#pragma once
#include "tcp_lattice.cuh"
#include "tcp_real.cuh"

namespace tcp {

template <typename real>
struct StepArgs {
    int nx, ny, nz;
    int ncell;                       // nx*ny*nz < 2^31
    int cell0, cell1;                // cells [cell0, cell1) are updated by this launch (the whole box, or the
                                     // boundary planes / the interior of a slab with ghost planes, tcp_step_begin)
    int aa;                          // streaming: 0 two-grid pull; AA in place: 1 even step, 2 odd step (tcp_step.cuh)
    int wall[3];                     // 1 = WALLS on that axis
    const real* h_in;  real* h_out;  // [27][N]
    const real* g_in;  real* g_out;  // [27][N]
    const real* f_in;  real* f_out;  // [QT][N] (thermal LB only)
    const real* phi_in; real* phi_out;
    const real* T_in;  real* T_out;
    real* u;                         // [3][N], updated in place (only read locally)
    const real* q_src;               // heat source or nullptr
    real* rk1_out; real* rk1_acc;    // Runge-Kutta paths with kappa_H = kappa_L: the fused kernel also does stage 1 (tcp_step.cuh,
    real rk1_c_out, rk1_c_acc;       // rk_stage1_local): Y1 = T^n + c_out R, accumulator = T^n + c_acc R (RK4); nullptr = off
    const real* wallT[3][2];         // wall-temperature planes
    real rho_L, drho, tau_L, dtau;   // eqs. 14, 22
    real xi, w_phi;                  // eq. 15; rate 1/(1/2 + 3M) (eq. 11, reading G3)
    real inv_xi;                     // 1 / xi (host-computed: two fp64 divisions per cell less)
    unsigned div_nx[3], div_ny[3];   // cell -> (x, y, z) without integer division: fast_div constants {m, s1, s2}
    unsigned div_hx[3];              // the same for nx / 2 (pair kernel)
    real sigma_ref, sigma_T, T_ref;  // eq. 9
    real sigma_TT;                   // parabolic sigma(T) (reading S19); 0 = eq. 9
    real kappa_L, dkappa, cp_L, dcp; // eqs. 23-24 (reading G5)
    real grav[3];                    // eq. 7
    real s_bulk, s_high, eps;
    int moving;                      // any wall velocity non-zero
    real wall_u[3][2][3];            // wall velocity [axis][face][component] (moving wall, reading S18)
    int wetting;                     // any wall with a contact angle other than 90 degrees
    real wet_a[3][2];                // a = -(2 / xi) cos(theta) of each wall (wetting boundary condition, reading S20); 0 = neutral
    int maxwell;                     // 1: Maxwellian (product-form) equilibria instead of the printed second-order ones (tcp_params::equilibrium)
    real eq_sigma;                   // 1 - maxwell: weight of the second-order polynomial equilibrium inside E (equilibrium_plus_half_force27)
    real cm_frame;                   // 1: central moments (about u); 0: raw moments (about the lattice at rest) = MRT (tcp_params::collision_space)
};

// packed pairs: the arrays are plain float arrays, the scalars are broadcast pairs
template <>
struct StepArgs<f32x2> {
    int nx, ny, nz;
    int ncell;
    int cell0, cell1;
    int aa;
    int wall[3];
    const float* h_in;  float* h_out;
    const float* g_in;  float* g_out;
    const float* f_in;  float* f_out;
    const float* phi_in; float* phi_out;
    const float* T_in;  float* T_out;
    float* u;
    const float* q_src;
    float* rk1_out; float* rk1_acc;
    f32x2 rk1_c_out, rk1_c_acc;
    const float* wallT[3][2];
    f32x2 rho_L, drho, tau_L, dtau;
    f32x2 xi, w_phi;
    f32x2 inv_xi;
    unsigned div_nx[3], div_ny[3], div_hx[3];
    f32x2 sigma_ref, sigma_T, T_ref;
    f32x2 sigma_TT;
    f32x2 kappa_L, dkappa, cp_L, dcp;
    f32x2 grav[3];
    f32x2 s_bulk, s_high, eps;
    int moving;
    float wall_u[3][2][3];
    int wetting;
    float wet_a[3][2];
    int maxwell;
    f32x2 eq_sigma, cm_frame;
    __host__ explicit StepArgs(const StepArgs<float>& A)
        : nx(A.nx), ny(A.ny), nz(A.nz), ncell(A.ncell), cell0(A.cell0), cell1(A.cell1), aa(A.aa), h_in(A.h_in), h_out(A.h_out), g_in(A.g_in), g_out(A.g_out),
          f_in(A.f_in), f_out(A.f_out), phi_in(A.phi_in), phi_out(A.phi_out), T_in(A.T_in), T_out(A.T_out), u(A.u), q_src(A.q_src), rk1_out(A.rk1_out), rk1_acc(A.rk1_acc), rk1_c_out(A.rk1_c_out), rk1_c_acc(A.rk1_c_acc),
          rho_L(A.rho_L), drho(A.drho), tau_L(A.tau_L), dtau(A.dtau), xi(A.xi), w_phi(A.w_phi), inv_xi(A.inv_xi), sigma_ref(A.sigma_ref),
          sigma_T(A.sigma_T), T_ref(A.T_ref), sigma_TT(A.sigma_TT), kappa_L(A.kappa_L), dkappa(A.dkappa), cp_L(A.cp_L), dcp(A.dcp),
          s_bulk(A.s_bulk), s_high(A.s_high), eps(A.eps), moving(A.moving), wetting(A.wetting), maxwell(A.maxwell), eq_sigma(A.eq_sigma), cm_frame(A.cm_frame) {
        for (int k = 0; k < 3; ++k) { div_nx[k] = A.div_nx[k]; div_ny[k] = A.div_ny[k]; div_hx[k] = A.div_hx[k]; }
        for (int a = 0; a < 3; ++a) {
            wall[a] = A.wall[a];
            grav[a] = f32x2(A.grav[a]);
            for (int f = 0; f < 2; ++f) {
                wallT[a][f] = A.wallT[a][f];
                wet_a[a][f] = A.wet_a[a][f];
                for (int k = 0; k < 3; ++k) wall_u[a][f][k] = A.wall_u[a][f][k];
            }
        }
    }
};

// ---------------------------------------------------------------------------------------------
// neighbourhood of one cell: element offsets to the 26 neighbours with periodic wrap, or, on a
// WALLS axis, clamped to the mirror cell (reading S9: walls half a cell outside the end cells)

// n / d for any 32-bit n, d >= 1 fixed per launch (Granlund-Montgomery round-up method): with l = ceil(log2 d),
// m = floor(2^32 (2^l - d) / d) + 1, s1 = min(l, 1), s2 = max(l - 1, 0):  q = (t + ((n - t) >> s1)) >> s2, t = mulhi(m, n).
// c = {m, s1, s2} comes from the host (fast_div_make in tcp_api.cu).
__device__ __forceinline__ unsigned fast_div(unsigned n, const unsigned c[3]) {
    const unsigned t = __umulhi(c[0], n);
    return (t + ((n - t) >> c[1])) >> c[2];
}

template <bool WALLS>
struct Nbh {
    int idx;
    int dx[3], dy[3], dz[3];         // offsets for c = -1, 0, +1
    bool lo[3], hi[3];               // WALLS: the cell touches the low / high wall of axis a
    int X[3], Y[3], Z[3];            // WALLS: coordinates of the wrapped / mirrored neighbours
    int nx, ny;

    // thread id -> cell: plain x, y, z order (a z-slab visiting order was measured 2-3 % slower)
    template <typename real>
    __device__ __forceinline__ void init(const StepArgs<real>& A, int cell) {
        const int t = (int)fast_div((unsigned)cell, A.div_nx), x = cell - t * A.nx;
        const int z = (int)fast_div((unsigned)t, A.div_ny), y = t - z * A.ny;
        init_xyz(A, x, y, z);
    }
    template <typename real>
    __device__ __forceinline__ void init_xyz(const StepArgs<real>& A, int x, int y, int z) {
        nx = A.nx; ny = A.ny;
        const int sy = A.nx, sz = A.nx * A.ny;
        idx = x + sy * y + sz * z;
        const bool wx = WALLS && A.wall[0], wy = WALLS && A.wall[1], wz = WALLS && A.wall[2];
        dx[1] = dy[1] = dz[1] = 0;
        dx[0] = x > 0 ? -1 : (wx ? 0 : A.nx - 1);
        dx[2] = x < A.nx - 1 ? 1 : (wx ? 0 : -(A.nx - 1));
        dy[0] = y > 0 ? -sy : (wy ? 0 : (A.ny - 1) * sy);
        dy[2] = y < A.ny - 1 ? sy : (wy ? 0 : -(A.ny - 1) * sy);
        dz[0] = z > 0 ? -sz : (wz ? 0 : (A.nz - 1) * sz);
        dz[2] = z < A.nz - 1 ? sz : (wz ? 0 : -(A.nz - 1) * sz);
        if (WALLS) {
            lo[0] = wx && x == 0; hi[0] = wx && x == A.nx - 1;
            lo[1] = wy && y == 0; hi[1] = wy && y == A.ny - 1;
            lo[2] = wz && z == 0; hi[2] = wz && z == A.nz - 1;
            X[1] = x; Y[1] = y; Z[1] = z;
            X[0] = x + dx[0]; X[2] = x + dx[2];
            Y[0] = y + dy[0] / sy; Y[2] = y + dy[2] / sy;
            Z[0] = z + dz[0] / sz; Z[2] = z + dz[2] / sz;
        }
    }
    __device__ __forceinline__ int at(int ox, int oy, int oz) const { return idx + dx[ox + 1] + dy[oy + 1] + dz[oz + 1]; }

    // first wall axis (x, then y, then z) crossed when stepping by (ox,oy,oz); -1 if none
    __device__ __forceinline__ int crossed(int ox, int oy, int oz, int& face) const {
        if (!WALLS) return -1;
        if (ox == -1 && lo[0]) { face = 0; return 0; }
        if (ox == 1 && hi[0]) { face = 1; return 0; }
        if (oy == -1 && lo[1]) { face = 0; return 1; }
        if (oy == 1 && hi[1]) { face = 1; return 1; }
        if (oz == -1 && lo[2]) { face = 0; return 2; }
        if (oz == 1 && hi[2]) { face = 1; return 2; }
        return -1;
    }
    // index into the tangential plane of wall `axis` at the neighbour (ox,oy,oz)
    __device__ __forceinline__ int tangential(int axis, int ox, int oy, int oz) const {
        const int xx = X[ox + 1], yy = Y[oy + 1], zz = Z[oz + 1];
        return axis == 0 ? zz * ny + yy : (axis == 1 ? zz * nx + xx : yy * nx + xx);
    }
};

template <typename real, bool WALLS>
__device__ __forceinline__ real wall_temperature(const StepArgs<real>& A, const Nbh<WALLS>& nb, int axis, int face,
                                                 int ox, int oy, int oz) {
    return A.wallT[axis][face][nb.tangential(axis, ox, oy, oz)];
}

// moving wall (reading S18): a population of direction (cx,cy,cz) that arrives at the cell
// from a wall moving with U_w is the bounced one plus 2 w (c . U_w) / c_s^2 (hydrodynamic lattice only;
// velocity-based model, no density factor).  (ox,oy,oz) = direction in which the wall lies (= -c).
template <typename real, bool WALLS, int QH = 27>
__device__ __forceinline__ real wall_velocity_term(const StepArgs<real>& A, const Nbh<WALLS>& nb, int q27i) {
    if (!WALLS || !A.moving) return real(0);
    const int cx = cx27(q27i), cy = cy27(q27i), cz = cz27(q27i);
    int face = 0;
    const int ax = nb.crossed(-cx, -cy, -cz, face);
    if (ax < 0) return real(0);
    const real* U = A.wall_u[ax][face];
    return real(6.0 * weight(QH, cls27(q27i))) * (real(cx) * U[0] + real(cy) * U[1] + real(cz) * U[2]);
}

// Wetting boundary condition (refs. [34], [35]; reading S20): ghost value of phi behind a wall with
// a = -(2 / xi) cos(theta), from the fluid cell phi_f across the wall:  n_w . grad phi = -(4 / xi) cos(theta) phi_w (1 - phi_w)
// with phi_w = (phi_f + phi_g) / 2 gives  a phi_w^2 - (1 + a) phi_w + phi_f = 0; the root that tends to phi_f for a -> 0,
// written without cancellation: phi_w = 2 phi_f / ((1 + a) + sqrt((1 + a)^2 - 4 a phi_f));  phi_g = 2 phi_w - phi_f.
// a = 0 returns phi_f exactly (the mirror ghost of S9).
template <typename scalar>
__device__ __forceinline__ scalar wetting_ghost(scalar a, scalar phi_f) {
    const scalar b = scalar(1) + a;
    const scalar phi_w = (scalar(2) * phi_f) / (b + sqrt(b * b - scalar(4) * a * phi_f));
    return scalar(2) * phi_w - phi_f;
}

// ---------------------------------------------------------------------------------------------
// isotropic finite differences with the D3Q27 weights (reading S3), evaluated as a tensor product:
//   grad_x = D_x S_y S_z,  lap = 6 (S_x S_y S_z - 1),   S = [1/6, 2/3, 1/6],  D = [-1/2, 0, 1/2]
// IS_TEMP: Dirichlet ghost 2 T_w - T(mirror); otherwise ghost = mirror cell (phi, neutral wetting).

// The 1/6 and 1/2 of S and D are applied once at the end: with s = m + 4c + p = 6 S and d = p - m = 2 D per direction,
//   grad_x = d_x s_y s_z / 72,   grad_y = s_x d_y s_z / 72,   grad_z = s_x s_y d_z / 72,   lap = s_x s_y s_z / 36 - 6 centre
// (52 flops instead of 82 with the factors applied at every level).
template <typename real, bool WALLS, bool IS_TEMP>
__device__ __forceinline__ void stencil27(const StepArgs<real>& A, const Nbh<WALLS>& nb, const real* __restrict__ psi,
                                          real& centre, real grad[3], real& lap) {
    const real four = real(4);
    real SS[3], DSy[3], SDx[3];
#pragma unroll
    for (int oz = -1; oz <= 1; ++oz) {
        real sx[3], dxv[3];
#pragma unroll
        for (int oy = -1; oy <= 1; ++oy) {
            real v[3];
#pragma unroll
            for (int ox = -1; ox <= 1; ++ox) {
                real t = __ldg(psi + nb.at(ox, oy, oz));
                if (WALLS && IS_TEMP) {
                    int face = 0;
                    const int ax = nb.crossed(ox, oy, oz, face);
                    if (ax >= 0) t = real(2) * wall_temperature(A, nb, ax, face, ox, oy, oz) - t;
                }
                if (WALLS && !IS_TEMP && A.wetting) {   // t is the mirror cell's value: first crossed wall in x, y, z order (S17)
                    int face = 0;
                    const int ax = nb.crossed(ox, oy, oz, face);
                    if (ax >= 0) t = wetting_ghost<real>(A.wet_a[ax][face], t);
                }
                v[ox + 1] = t;
            }
            if (oy == 0 && oz == 0) centre = v[1];
            sx[oy + 1] = (v[0] + v[2]) + four * v[1];
            dxv[oy + 1] = v[2] - v[0];
        }
        SS[oz + 1] = (sx[0] + sx[2]) + four * sx[1];
        DSy[oz + 1] = sx[2] - sx[0];
        SDx[oz + 1] = (dxv[0] + dxv[2]) + four * dxv[1];
    }
    const real c72 = real(1.0 / 72.0);
    grad[0] = c72 * ((SDx[0] + SDx[2]) + four * SDx[1]);
    grad[1] = c72 * ((DSy[0] + DSy[2]) + four * DSy[1]);
    grad[2] = c72 * (SS[2] - SS[0]);
    lap = real(1.0 / 36.0) * ((SS[0] + SS[2]) + four * SS[1]) - real(6) * centre;
}

// ---------------------------------------------------------------------------------------------
// pulls (two-grid): a_q(x) = a~_q(x - c_q); halfway bounce-back a~_opp(x) for h, g;
// anti-bounce-back -f~_opp(x) + 2 w T_w for f (reading S9)

template <typename real, bool WALLS>
__device__ __forceinline__ void pull27(const StepArgs<real>& A, const Nbh<WALLS>& nb, const real* __restrict__ a, real out[27]) {
    const long long N = A.ncell;
#pragma unroll
    for (int q = 0; q < 27; ++q) {
        const int cx = cx27(q), cy = cy27(q), cz = cz27(q);
        int face = 0;
        if (WALLS && nb.crossed(-cx, -cy, -cz, face) >= 0)
            out[q] = a[(26 - q) * N + nb.idx];
        else
            out[q] = a[q * N + nb.at(-cx, -cy, -cz)];
    }
}

template <typename real, int Q, bool WALLS>
__device__ __forceinline__ void pull_thermal(const StepArgs<real>& A, const Nbh<WALLS>& nb, const real* __restrict__ a, real out[Q]) {
    const long long N = A.ncell;
    static_for<0, Q>([&](auto K) {
        constexpr int k = decltype(K)::value, q = q_of(Q, k);
        constexpr int cx = cx27(q), cy = cy27(q), cz = cz27(q);
        int face = 0;
        const int ax = nb.crossed(-cx, -cy, -cz, face);
        if (WALLS && ax >= 0)
            out[k] = real(2.0 * weight(Q, cls27(q))) * wall_temperature(A, nb, ax, face, -cx, -cy, -cz)
                     - a[(Q - 1 - k) * N + nb.idx];
        else
            out[k] = a[k * N + nb.at(-cx, -cy, -cz)];
    });
}

// ---------------------------------------------------------------------------------------------
// raw moments of a D3Q27 population set up to order 2, by successive sums along x, y, z

template <typename real>
struct Mom2 {
    real m0, mx, my, mz, mxx, myy, mzz, mxy, mxz, myz;
};

template <typename real, bool SECOND>
__device__ __forceinline__ Mom2<real> moments27(const real a[27]) {
    Mom2<real> M;
    real t00[3], t01[3], t02[3], t10[3], t11[3], t20[3];
#pragma unroll
    for (int z = 0; z < 3; ++z) {
        real s0[3], s1[3], s2[3];
#pragma unroll
        for (int y = 0; y < 3; ++y) {
            const real m = a[9 * z + 3 * y], c = a[9 * z + 3 * y + 1], p = a[9 * z + 3 * y + 2];
            s2[y] = p + m;
            s0[y] = s2[y] + c;
            s1[y] = p - m;
        }
        t00[z] = (s0[0] + s0[2]) + s0[1];
        t01[z] = s0[2] - s0[0];
        t10[z] = (s1[0] + s1[2]) + s1[1];
        if (SECOND) {
            t02[z] = s0[0] + s0[2];
            t11[z] = s1[2] - s1[0];
            t20[z] = (s2[0] + s2[2]) + s2[1];
        }
    }
    M.m0 = (t00[0] + t00[2]) + t00[1];
    M.mz = t00[2] - t00[0];
    M.my = (t01[0] + t01[2]) + t01[1];
    M.mx = (t10[0] + t10[2]) + t10[1];
    if (SECOND) {
        M.mzz = t00[0] + t00[2];
        M.myz = t01[2] - t01[0];
        M.myy = (t02[0] + t02[2]) + t02[1];
        M.mxz = t10[2] - t10[0];
        M.mxy = (t11[0] + t11[2]) + t11[1];
        M.mxx = (t20[0] + t20[2]) + t20[1];
    } else {
        M.mxx = M.myy = M.mzz = M.mxy = M.mxz = M.myz = real(0);
    }
    return M;
}

// ---------------------------------------------------------------------------------------------
// 1-D inverse central-moment columns on {-1, 0, +1}: r_k(c; u) is the population with k-th
// central moment 1 and the other two 0
template <typename real>
struct R1D {
    real r0[3], r1[3];   // index c+1; r2 = {1/2, -1, 1/2} is constant
    __device__ __forceinline__ void set(real u) {
        const real uu = u * u, hu = real(0.5) * u;
        r0[0] = real(0.5) * uu - hu; r0[1] = real(1) - uu; r0[2] = real(0.5) * uu + hu;
        r1[0] = u - real(0.5);       r1[1] = real(-2) * u; r1[2] = u + real(0.5);
    }
};

// E_q = w_q [ A0 + 3 c.v + 4.5 (c.u)(c.b) ]  -- equilibrium (eq. 12 or eq. 18) plus half the Guo
// force populations (ref. [20]), merged:
//   scalar (h, f):  A0 = s - 1.5 u.b,  v = s u + a/2,  b = s u + a
//   hydro  (g):     A0 = p* - 1.5 u.b, v = u + a/2,    b = u + a
// Q = 27, or 19 (D3Q19 hydrodynamic lattice: its weights, the eight corner entries of out[] are set to 0).
template <typename real, int Q = 27>
__device__ __forceinline__ void equilibrium_plus_half_force27(real A0, const real u[3], const real v[3], const real b[3], real out[27]) {
#pragma unroll
    for (int q = 0; q < 13; ++q) {
        const int cx = cx27(q), cy = cy27(q), cz = cz27(q);
        if (!has_class(Q, cls27(q))) { out[q] = real(0); out[26 - q] = real(0); continue; }
        const real w = real(weight(Q, cls27(q)));
        const real cu = real(cx) * u[0] + real(cy) * u[1] + real(cz) * u[2];
        const real cb = real(cx) * b[0] + real(cy) * b[1] + real(cz) * b[2];
        const real cv = real(cx) * v[0] + real(cy) * v[1] + real(cz) * v[2];
        const real sym = w * (A0 + real(4.5) * cu * cb);
        const real asym = real(3) * w * cv;
        out[q] = sym + asym;
        out[26 - q] = sym - asym;
    }
    out[13] = real(weight(Q, 0)) * A0;
}

// Maxwellian equilibrium (tcp_params::equilibrium = TCP_EQ_MAXWELLIAN): the continuous Maxwell-Boltzmann distribution in
// central-moment space on D3Q27 is the product form  s prod_axis p(c_a; u_a),  p(0; u) = 2/3 - u^2 = w(0) (1 - 3/2 u^2),
// p(+-1; u) = 1/6 +- u/2 + u^2/2 = w(1) (1 +- 3 u + 3 u^2)  (central moments 1, 0, 1/3 per axis).  Its moments up to second
// order are those of the printed equilibria (eqs. 12, 18), so the relaxed moments of the closed-form collisions do not
// change; only these populations replace the polynomial ones.   out_q += s w_q pi_x pi_y pi_z.
// DEV: out_q += s w_q (pi_x pi_y pi_z - 1) -- the form the hydrodynamic populations need (eq. 18 subtracts w_q), evaluated
// without ever forming the 1: with pi = 1 + d, d(0) = -3/2 u^2, d(+-1) = +-3u + 3u^2,
//   pi_x pi_y - 1 = d_x + d_y + d_x d_y =: t,   pi_x pi_y pi_z - 1 = t + d_z + t d_z,
// so that g~ stays a deviation of size O(u) also in single precision (w_q (p* - 1) + product would cancel to ~1e-4 relative).
template <typename real, bool DEV>
__device__ __forceinline__ void add_product_form27(real s, const real u[3], real out[27]) {
    real d[3][3];   // [axis][c + 1]
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const real uu3 = real(3) * u[a] * u[a], u3 = real(3) * u[a];
        d[a][1] = real(-0.5) * uu3;
        d[a][0] = uu3 - u3;
        d[a][2] = uu3 + u3;
    }
    real t[3][3];   // [cy][cx]: pi_x pi_y - 1
#pragma unroll
    for (int y = 0; y < 3; ++y)
#pragma unroll
        for (int x = 0; x < 3; ++x) t[y][x] = (d[0][x] + d[1][y]) + d[0][x] * d[1][y];
#pragma unroll
    for (int z = 0; z < 3; ++z)
#pragma unroll
        for (int y = 0; y < 3; ++y)
#pragma unroll
            for (int x = 0; x < 3; ++x) {
                const int q = 9 * z + 3 * y + x;
                const real dev = (t[y][x] + d[2][z]) + t[y][x] * d[2][z];
                const real sw = s * real(weight(27, cls27(q)));
                out[q] += DEV ? sw * dev : sw + sw * dev;
            }
}

// out_q += sum_alpha m_alpha R^alpha_q(u): populations whose first-order central moments are m and
// whose other central moments vanish (tensor-product monomial basis of D3Q27, reading S2)
template <typename real>
__device__ __forceinline__ void add_first_order27(const real m[3], const R1D<real>& rx, const R1D<real>& ry, const R1D<real>& rz, real out[27]) {
    real P[3][3], W[3][3];   // [cy][cx]
#pragma unroll
    for (int y = 0; y < 3; ++y)
#pragma unroll
        for (int x = 0; x < 3; ++x) {
            P[y][x] = m[0] * rx.r1[x] * ry.r0[y] + m[1] * rx.r0[x] * ry.r1[y];
            W[y][x] = m[2] * rx.r0[x] * ry.r0[y];
        }
#pragma unroll
    for (int z = 0; z < 3; ++z)
#pragma unroll
        for (int y = 0; y < 3; ++y)
#pragma unroll
            for (int x = 0; x < 3; ++x) out[9 * z + 3 * y + x] += rz.r0[z] * P[y][x] + rz.r1[z] * W[y][x];
}

// out_q += sum_{alpha<=beta} A_{alpha beta} R^{alpha beta}_q(u): second-order central moments
template <typename real>
__device__ __forceinline__ void add_second_order27(real Axx, real Ayy, real Azz, real Axy, real Axz, real Ayz, const R1D<real>& rx,
                                                   const R1D<real>& ry, const R1D<real>& rz, real out[27]) {
    const real r2[3] = {real(0.5), real(-1), real(0.5)};
    real P[3][3], Qm[3][3], W[3][3];
#pragma unroll
    for (int y = 0; y < 3; ++y)
#pragma unroll
        for (int x = 0; x < 3; ++x) {
            P[y][x] = Axx * r2[x] * ry.r0[y] + Ayy * rx.r0[x] * r2[y] + Axy * rx.r1[x] * ry.r1[y];
            Qm[y][x] = Axz * rx.r1[x] * ry.r0[y] + Ayz * rx.r0[x] * ry.r1[y];
            W[y][x] = Azz * rx.r0[x] * ry.r0[y];
        }
#pragma unroll
    for (int z = 0; z < 3; ++z)
#pragma unroll
        for (int y = 0; y < 3; ++y)
#pragma unroll
            for (int x = 0; x < 3; ++x)
                out[9 * z + 3 * y + x] += rz.r0[z] * P[y][x] + rz.r1[z] * Qm[y][x] + r2[z] * W[y][x];
}

// D3Q19 (hydrodynamic lattice, basis of reading S2: the monomials x^a y^b z^c, a, b, c <= 2, abc = 0):
// out_q += populations whose second-order central moments are A_{alpha beta} and whose other basis central moments
// vanish.  Their raw moments over the basis are M_b = 1/2 sum_{alpha beta} A_{alpha beta} d_alpha d_beta b (u) (Taylor
// expansion of b(u + xi); the derivatives of a basis monomial are basis monomials, so no uncontrolled moment enters):
//   x_a^2: A_aa;  x_a x_b: A_ab;  x_a^2 x_b: A_aa u_b + 2 A_ab u_a;  x_a^2 x_b^2: A_aa u_b^2 + A_bb u_a^2 + 4 A_ab u_a u_b,
// and the populations follow from the lattice's raw-moment inversion (rest, 6 axis, 12 diagonal velocities), the same
// one add_first_order_thermal<19> uses.  Entries of out[] at the eight corner velocities are left untouched.
template <typename real>
__device__ __forceinline__ void add_second_order19(real Axx, real Ayy, real Azz, real Axy, real Axz, real Ayz, const real u[3], real out[27]) {
    const real Ad[3] = {Axx, Ayy, Azz}, Ao[3] = {Axy, Axz, Ayz};   // pair index p: 0 = (x,y), 1 = (x,z), 2 = (y,z)
    real m22[3], m12[3], m21[3];
#pragma unroll
    for (int p = 0; p < 3; ++p) {
        const int a = (p == 2 ? 1 : 0), b = (p == 0 ? 1 : 2);
        m21[p] = Ad[a] * u[b] + real(2) * Ao[p] * u[a];                                  // x_a^2 x_b
        m12[p] = Ad[b] * u[a] + real(2) * Ao[p] * u[b];                                  // x_a x_b^2
        m22[p] = Ad[a] * u[b] * u[b] + Ad[b] * u[a] * u[a] + real(4) * Ao[p] * u[a] * u[b];
    }
    out[13] += -(Axx + Ayy + Azz) + (m22[0] + m22[1] + m22[2]);
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        // the two pairs containing axis a and, in each, the moment of x_a x_other^2
        const int p1 = (a == 2 ? 1 : 0), p2 = (a == 0 ? 1 : 2);
        const real q1 = (a == 0) ? m12[0] : (a == 1 ? m21[0] : m21[1]);
        const real q2 = (a == 0) ? m12[1] : (a == 1 ? m12[2] : m21[2]);
        const real sym = real(0.5) * (Ad[a] - m22[p1] - m22[p2]), asym = real(-0.5) * (q1 + q2);
        const int qp = 13 + (a == 0 ? 1 : (a == 1 ? 3 : 9));
        out[qp] += sym + asym;
        out[26 - qp] += sym - asym;
    }
#pragma unroll
    for (int p = 0; p < 3; ++p) {
        const int a = (p == 2 ? 1 : 0), b = (p == 0 ? 1 : 2);
        const int sa = (a == 0 ? 1 : 3), sb = (b == 1 ? 3 : 9);                          // index strides of the two axes
#pragma unroll
        for (int ca = -1; ca <= 1; ca += 2)
#pragma unroll
            for (int cb = -1; cb <= 1; cb += 2)
                out[13 + ca * sa + cb * sb] += real(0.25) * (m22[p] + real(ca) * m12[p] + real(cb) * m21[p] + real(ca * cb) * Ao[p]);
    }
}

}  // namespace tcp
