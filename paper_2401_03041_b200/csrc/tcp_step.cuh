// The kernels proper (see tcp_kernels.cuh for the overview).
#pragma once
#include "tcp_kernels.cuh"

namespace tcp {

// MODE of the collision templates: 0 closed-form central moments (or raw moments, StepArgs::cm_frame), 1 BGK, 2 general rates,
// 3 roofline calibration (no collision), 4 = mode 0 with the Maxwellian equilibrium (D3Q27 lattices; a compile-time mode
// because a run-time branch around the product form cost the fp32 pair kernel 2.2 % and the fp64 D3Q27 kernel 1.6 %)
template <int MODE> __host__ __device__ constexpr bool mode_maxwell() { return MODE == 4; }

#ifndef TCP_BLOCK
#define TCP_BLOCK 128
#endif
// 3 resident blocks of 128 threads per SM (168 registers per thread, ~90 B of spills in fp64) measured
// 5 % faster than 2 blocks at 248 registers; 4 blocks (128 registers) spill too much (profiles/).
#ifndef TCP_MINB
#define TCP_MINB 3
#endif
constexpr int kBlock = TCP_BLOCK;

// fp32 only.  In real arithmetic the collision conserves the zeroth moment (sum_q E_q = s because
// sum_q w_q = 1), but the rounded weights do not sum to 1, which re-creates the whole population
// with the same relative bias (~1e-8) every step: sum(phi) then drifts linearly (measured 7.5e-5
// over 1e4 steps).  So the rest population is not taken from the formula but written as a remainder.
// Round 1 summed the zeroth moment and the remainder in fp64 (252 conversions + 238 DADD per pair of
// cells: 15 % of the pair kernel's instructions, XU pipe 31 % busy; TCP_F32_EXACT0 = 1 restores it).
// Now both stay in fp32 and are built from the SAME ordered partial sum over the 26 moving populations,
//     s = fl(P_in + a_rest),   a~_rest = fl(s - P_out),   P = ((a_0 + a_26) + (a_1 + a_25)) + ...,
// so that wherever the state is steady (a~_q = a_q for the moving q, hence P_out = P_in) the remainder
// reproduces itself exactly (s / 2 <= P <= 2 s: the subtraction is exact, Sterbenz) and the stored total stops
// changing.  With the remainder taken against a differently ordered sum (e.g. the tree of moments27)
// every quasi-steady cell repeats the same rounding mismatch step after step and sum(phi) drifts
// 1.5e-6 over 1e4 steps (measured).  In fp64 the bias is ~1e-17 per step and the arithmetic is left as derived.
#ifndef TCP_F32_EXACT0
#define TCP_F32_EXACT0 0
#endif
template <typename real>
__device__ __forceinline__ wide_t<real> exact_sum27(const real a[27]) {
    wide_t<real> s = wide_zero<real>();
#pragma unroll
    for (int q = 0; q < 27; ++q) s += widen(a[q]);
    return s;
}
// P of the comment above
template <typename real>
__device__ __forceinline__ real moving_sum27(const real a[27]) {
    real P = a[0] + a[26];
#pragma unroll
    for (int q = 1; q < 13; ++q) P += (a[q] + a[26 - q]);
    return P;
}
template <typename real>
__device__ __forceinline__ void conserve_zeroth27(real a[27], real s, wide_t<real> s_exact) {
    if constexpr (real_traits<real>::single) {
        if constexpr (TCP_F32_EXACT0) {
#pragma unroll
            for (int q = 0; q < 27; ++q)
                if (q != 13) s_exact -= widen(a[q]);
            a[13] = narrow<real>(s_exact);
        } else {
            a[13] = s - moving_sum27<real>(a);
        }
    }
}

// In-place central-moment transform of a D3Q27 population set indexed 9 c_z + 3 c_y + c_x (+13):
// forward: populations -> kappa_{abc} stored at 9c + 3b + a; inverse: back.  Three sweeps of the
// 1-D transform on {-1, 0, 1}:  k0 = sum p, k1 = sum (c - u) p, k2 = sum (c - u)^2 p.
template <typename real, bool FORWARD>
__device__ __forceinline__ void central_transform27(real X[27], const real u[3]) {
#pragma unroll
    for (int pass = 0; pass < 3; ++pass) {
        const int axis = FORWARD ? pass : 2 - pass;
        const int stride = axis == 0 ? 1 : (axis == 1 ? 3 : 9);
        const real ua = u[axis], uu = ua * ua;
#pragma unroll
        for (int j = 0; j < 9; ++j) {
            // base index of the j-th line along `axis`
            const int base = axis == 0 ? 3 * j : (axis == 1 ? (j / 3) * 9 + (j % 3) : j);
            real& e0 = X[base]; real& e1 = X[base + stride]; real& e2 = X[base + 2 * stride];
            if (FORWARD) {
                const real m = e0, c = e1, p = e2;
                const real m0 = (m + p) + c, m1 = p - m, m2 = p + m;
                e0 = m0;
                e1 = m1 - ua * m0;
                e2 = m2 - real(2) * ua * m1 + uu * m0;
            } else {
                const real k0 = e0, k1 = e1, k2 = e2;
                const real m1 = k1 + ua * k0, m2 = k2 + real(2) * ua * k1 + uu * k0;
                e0 = real(0.5) * (m2 - m1);
                e1 = k0 - m2;
                e2 = real(0.5) * (m2 + m1);
            }
        }
    }
}

// ---- phase-field LB on one cell: eqs. 10-15 ---------------------------------------------------
// h = pulled populations; G = grad phi^n, phi_c = phi^n (interface force from the stored phi,
// reading S10); un = u^n.  Writes h~ and phi' = sum h (eq. 13).
template <typename real, int MODE>
__device__ __forceinline__ real collide_phase(const StepArgs<real>& A, real h[27], const real G[3], real phi_c, const real un[3]) {
    const Mom2<real> M = moments27<real, false>(h);
    wide_t<real> phin_exact = wide_zero<real>();
    real phin = M.m0;
    if constexpr (real_traits<real>::single) {
        if constexpr (TCP_F32_EXACT0) { phin_exact = exact_sum27<real>(h); phin = narrow<real>(phin_exact); }
        else phin = moving_sum27<real>(h) + h[13];
    }
    // a = c_s^2 [4 phi (1 - phi) / xi] n,  n = G / sqrt(G.G + eps)   (eq. 15, readings S7, S8)
    const real inv = rsqrt_<real>(G[0] * G[0] + G[1] * G[1] + G[2] * G[2] + A.eps);
    const real mag = real(4.0 / 3.0) * phi_c * (real(1) - phi_c) * A.inv_xi * inv;
    real a[3] = {mag * G[0], mag * G[1], mag * G[2]};
    const real w = A.w_phi;
    if (MODE == 1) {   // a~ = (1-w) a + w [a_eq + F(a (2-w)/w)/2]
        const real sc = (real(2) - w) / w;
        a[0] *= sc; a[1] *= sc; a[2] *= sc;
    }
    real b[3], v[3];
#pragma unroll
    // E = sigma h_eq(eq. 12) + F/2; sigma = 1, or 0 with the Maxwellian equilibrium, whose product form is added instead
    const real se = mode_maxwell<MODE>() ? real(0) : phin;
    for (int al = 0; al < 3; ++al) { b[al] = se * un[al] + a[al]; v[al] = se * un[al] + real(0.5) * a[al]; }
    const real A0 = se - real(1.5) * (un[0] * b[0] + un[1] * b[1] + un[2] * b[2]);
    real out[27];
    equilibrium_plus_half_force27<real>(A0, un, v, b, out);
    if constexpr (mode_maxwell<MODE>()) add_product_form27<real, false>(phin, un, out);
    if (MODE == 1) {
#pragma unroll
        for (int q = 0; q < 27; ++q) h[q] = (real(1) - w) * h[q] + w * out[q];
    } else {
        // first-order central moments of (h - h_eq) + F/2 relax with w_phi, everything else with 1
        const real k1 = real(1) - w;
        const real m[3] = {k1 * ((M.mx - phin * un[0]) + real(0.5) * a[0]),
                           k1 * ((M.my - phin * un[1]) + real(0.5) * a[1]),
                           k1 * ((M.mz - phin * un[2]) + real(0.5) * a[2])};
        // the populations that carry the relaxed moments: central moments about u, or, for the raw-moment (MRT) space, about
        // the lattice at rest.  The relaxed amplitudes are the same in both spaces: (h - h_eq) + F/2 has no zeroth moment, so
        // its first central and raw moments coincide
        R1D<real> rx, ry, rz;
        rx.set(A.cm_frame * un[0]); ry.set(A.cm_frame * un[1]); rz.set(A.cm_frame * un[2]);
        add_first_order27<real>(m, rx, ry, rz, out);
#pragma unroll
        for (int q = 0; q < 27; ++q) h[q] = out[q];
    }
    conserve_zeroth27<real>(h, phin, phin_exact);
    return phin;
}

// ---- hydrodynamic LB on one cell: eqs. 16-22, forces of eqs. 7-9 -------------------------------
// g = pulled populations; phi_c, G, lapPhi from phi^n (S16); T_c, Th = grad T^n.  Writes g~, u^{n+1}.
// QH = 27 or 19 (D3Q19 hydrodynamic lattice): g[] stays indexed as D3Q27 with the eight corner entries 0.
template <typename real, int MODE, int QH = 27>
__device__ __forceinline__ void collide_hydro(const StepArgs<real>& A, real g[27], real phi_c, const real G[3], real lapPhi,
                                              real T_c, const real Th[3], real u[3]) {
    const Mom2<real> M = moments27<real, true>(g);
    wide_t<real> ps_exact = wide_zero<real>();
    real ps = M.m0;                                         // p* (eq. 17)
    if constexpr (real_traits<real>::single) {
        if constexpr (TCP_F32_EXACT0) { ps_exact = exact_sum27<real>(g); ps = narrow<real>(ps_exact); }
        else ps = moving_sum27<real>(g) + g[13];
    }
    const real j[3] = {M.mx, M.my, M.mz};
    const real rho = A.rho_L + phi_c * A.drho;              // eq. 14
    const real tau = A.tau_L + phi_c * A.dtau;              // eq. 22
    // eq. 9 plus the parabolic term of reading S19; dsigma = d sigma / dT carries the Marangoni term of eq. 8
    const real dTr = T_c - A.T_ref;
    const real dsigma = A.sigma_T + A.sigma_TT * dTr;
    const real sigma = A.sigma_ref + A.sigma_T * dTr + real(0.5) * A.sigma_TT * dTr * dTr;
    // mu_phi = 4 beta phi (phi-1)(phi-1/2) - k lap phi, beta = 12 sigma/xi, k = 3 sigma xi/2  (S5)
    const real mu = real(48) * sigma * A.inv_xi * phi_c * (phi_c - real(1)) * (phi_c - real(0.5)) - real(1.5) * sigma * A.xi * lapPhi;
    const real GG = G[0] * G[0] + G[1] * G[1] + G[2] * G[2];
    const real TG = Th[0] * G[0] + Th[1] * G[1] + Th[2] * G[2];
    const real mar = real(1.5) * A.xi * dsigma;             // eq. 8 (with |grad phi|^2, G2)
    const real pcoef = ps * real(1.0 / 3.0) * A.drho;       // eq. 20
    const real i2r = real(0.5) / rho;
    real F[3], us[3];
#pragma unroll
    for (int al = 0; al < 3; ++al) {
        F[al] = mu * G[al] + mar * (GG * Th[al] - TG * G[al]) + rho * A.grav[al] - pcoef * G[al];
        us[al] = j[al] + F[al] * i2r;                       // predictor u* (S4)
    }
    const real om = real(1) / (tau + real(0.5));
    {   // F_mu = -(tau/(tau+1/2)) (rho_H - rho_L) Pi* . G, Pi* = sum c c (g - g_eq(p*, u*))  (eq. 21)
        const real p3 = ps * real(1.0 / 3.0);
        const real Pxx = M.mxx - (p3 + us[0] * us[0]), Pyy = M.myy - (p3 + us[1] * us[1]), Pzz = M.mzz - (p3 + us[2] * us[2]);
        const real Pxy = M.mxy - us[0] * us[1], Pxz = M.mxz - us[0] * us[2], Pyz = M.myz - us[1] * us[2];
        const real cf = -(tau * om) * A.drho;
        F[0] += cf * (Pxx * G[0] + Pxy * G[1] + Pxz * G[2]);
        F[1] += cf * (Pxy * G[0] + Pyy * G[1] + Pyz * G[2]);
        F[2] += cf * (Pxz * G[0] + Pyz * G[1] + Pzz * G[2]);
    }
    real a[3], d[3];
#pragma unroll
    for (int al = 0; al < 3; ++al) {
        d[al] = -F[al] * i2r;                               // j - u
        u[al] = j[al] + F[al] * i2r;                        // u^{n+1} (S6)
        a[al] = real(2) * F[al] * i2r;                      // Guo vector F / rho
    }
    if (MODE == 1) {
        const real sc = (real(2) - om) / om;
        a[0] *= sc; a[1] *= sc; a[2] *= sc;
    }
    real b[3], v[3];
#pragma unroll
    // E = w_q p* + sigma w_q [poly(u) of eq. 18] + F/2; Maxwellian (sigma = 0): + w_q (pi_x pi_y pi_z - 1) instead of w_q poly(u)
    const real sg = mode_maxwell<MODE>() ? real(0) : real(1);
    for (int al = 0; al < 3; ++al) { b[al] = sg * u[al] + a[al]; v[al] = sg * u[al] + real(0.5) * a[al]; }
    const real A0 = ps - real(1.5) * (u[0] * b[0] + u[1] * b[1] + u[2] * b[2]);
    real out[27];
    equilibrium_plus_half_force27<real, QH>(A0, u, v, b, out);
    if constexpr (mode_maxwell<MODE>()) add_product_form27<real, true>(real(1), u, out);
    if (MODE == 1) {
#pragma unroll
        for (int q = 0; q < 27; ++q) g[q] = (real(1) - om) * g[q] + om * out[q];
    } else if (MODE == 2) {
        static_assert(MODE != 2 || QH == 27, "general central-moment rates: the sweep transform exists for the tensor-product D3Q27 basis only");
        // general rates (s_high != 1): g~ = E + K^-1 (I - S) K X,  X = (g - g_eq) + F/2 = g - E(-a)
        // (I - S vanishes on orders 0 and 1).  K is applied as three sweeps of the 1-D central-moment
        // transform (x, y, z), its inverse as the reverse sweeps.
        real X[27];
        {
            real bm[3], vm[3];
#pragma unroll
            for (int al = 0; al < 3; ++al) { bm[al] = sg * u[al] - a[al]; vm[al] = sg * u[al] - real(0.5) * a[al]; }
            equilibrium_plus_half_force27<real, QH>(ps - real(1.5) * (u[0] * bm[0] + u[1] * bm[1] + u[2] * bm[2]), u, vm, bm, X);
#pragma unroll
            for (int q = 0; q < 27; ++q) X[q] = g[q] - X[q];
        }
        const real uf[3] = {A.cm_frame * u[0], A.cm_frame * u[1], A.cm_frame * u[2]};   // raw-moment space: transform about rest
        central_transform27<real, true>(X, uf);
        const real k2 = real(1) - om, k3 = real(1) - A.s_high;
        const real tr3 = (X[2] + X[6] + X[18]) * real(1.0 / 3.0), kb = (real(1) - A.s_bulk) * tr3;
#pragma unroll
        for (int q = 0; q < 27; ++q) {
            const int order = (q % 3) + (q / 3) % 3 + q / 9;
            if (order <= 1) X[q] = real(0);
            else if (order == 2) X[q] = (q == 2 || q == 6 || q == 18) ? k2 * (X[q] - tr3) + kb : k2 * X[q];
            else X[q] = k3 * X[q];
        }
        central_transform27<real, false>(X, uf);
#pragma unroll
        for (int q = 0; q < 27; ++q) g[q] = out[q] + X[q];
    } else {
        // second-order central moments of g - g_eq: deviatoric part relaxes with omega, trace with
        // s_bulk, everything else with 1 (reading S2); Guo populations have none
        const real p3 = ps * real(1.0 / 3.0);
        real kxx = M.mxx - (p3 + u[0] * u[0]) - real(2) * u[0] * d[0];
        real kyy = M.myy - (p3 + u[1] * u[1]) - real(2) * u[1] * d[1];
        real kzz = M.mzz - (p3 + u[2] * u[2]) - real(2) * u[2] * d[2];
        const real kxy = M.mxy - u[0] * u[1] - u[0] * d[1] - u[1] * d[0];
        const real kxz = M.mxz - u[0] * u[2] - u[0] * d[2] - u[2] * d[0];
        const real kyz = M.myz - u[1] * u[2] - u[1] * d[2] - u[2] * d[1];
        const real tr3 = (kxx + kyy + kzz) * real(1.0 / 3.0);
        const real k2 = real(1) - om, kb = (real(1) - A.s_bulk) * tr3;
        kxx = k2 * (kxx - tr3) + kb; kyy = k2 * (kyy - tr3) + kb; kzz = k2 * (kzz - tr3) + kb;
        // (g - g_eq) + F/2 has neither a zeroth nor a first moment, so its second central and raw moments coincide; only the
        // populations that carry them differ between the central-moment and the raw-moment (MRT) space
        const real uf[3] = {A.cm_frame * u[0], A.cm_frame * u[1], A.cm_frame * u[2]};
        if constexpr (QH == 27) {
            R1D<real> rx, ry, rz;
            rx.set(uf[0]); ry.set(uf[1]); rz.set(uf[2]);
            add_second_order27<real>(kxx, kyy, kzz, k2 * kxy, k2 * kxz, k2 * kyz, rx, ry, rz, out);
        } else {
            add_second_order19<real>(kxx, kyy, kzz, k2 * kxy, k2 * kxz, k2 * kyz, uf, out);
        }
#pragma unroll
        for (int q = 0; q < 27; ++q) g[q] = out[q];
    }
    conserve_zeroth27<real>(g, ps, ps_exact);
}

// ---- thermal LB on one cell: eqs. 27-29 (rho c_p = 1 on this path, S11) ------------------------
template <typename real, int Q, int MODE>
__device__ __forceinline__ real collide_thermal(const StepArgs<real>& A, real f[Q], real phi_new, const real u[3], real qT) {
    real Tn = real(0), j[3] = {real(0), real(0), real(0)};
    wide_t<real> Tn_exact = wide_zero<real>();
    constexpr bool ordered = real_traits<real>::single && !TCP_F32_EXACT0;   // see conserve_zeroth27
    if constexpr (ordered) {
        static_for<0, Q / 2>([&](auto K) { constexpr int k = decltype(K)::value; Tn += (f[k] + f[Q - 1 - k]); });
        Tn += f[Q / 2];
    }
    static_for<0, Q>([&](auto K) {
        constexpr int k = decltype(K)::value, q = q_of(Q, k);
        if constexpr (real_traits<real>::single && TCP_F32_EXACT0) Tn_exact += widen(f[k]); else
        if constexpr (!ordered) Tn += f[k];                  // eq. 28
        if constexpr (cx27(q) != 0) j[0] += real(cx27(q)) * f[k];
        if constexpr (cy27(q) != 0) j[1] += real(cy27(q)) * f[k];
        if constexpr (cz27(q) != 0) j[2] += real(cz27(q)) * f[k];
    });
    if constexpr (real_traits<real>::single && TCP_F32_EXACT0) Tn = narrow<real>(Tn_exact);
    const real kap = A.kappa_L + phi_new * A.dkappa;         // eq. 23 (G5)
    const real w = real(1) / (real(0.5) + real(3) * kap);    // eq. 29 read as a rate (G4)
    real out[Q];
    if constexpr (Q == 27 && mode_maxwell<MODE>()) {
#pragma unroll
        for (int q = 0; q < 27; ++q) out[q] = real(0);
        add_product_form27<real, false>(Tn, u, out);
    } else thermal_equilibrium<real, Q>(Tn, u, out);
    if (MODE == 1) {
        static_for<0, Q>([&](auto K) { constexpr int k = decltype(K)::value; out[k] = (real(1) - w) * f[k] + w * out[k]; });
    } else {
        const real k1 = real(1) - w;
        const real m[3] = {k1 * (j[0] - Tn * u[0]), k1 * (j[1] - Tn * u[1]), k1 * (j[2] - Tn * u[2])};
        const real uf[3] = {A.cm_frame * u[0], A.cm_frame * u[1], A.cm_frame * u[2]};   // see collide_phase
        if constexpr (Q == 27) {
            R1D<real> rx, ry, rz;
            rx.set(uf[0]); ry.set(uf[1]); rz.set(uf[2]);
            add_first_order27<real>(m, rx, ry, rz, out);
        } else {
            add_first_order_thermal<real, Q>(m, uf, out);
        }
    }
    if constexpr (real_traits<real>::single) {   // see conserve_zeroth27
        if constexpr (TCP_F32_EXACT0) {
            wide_t<real> rest = Tn_exact;
            static_for<0, Q>([&](auto K) { constexpr int k = decltype(K)::value; if constexpr (k != Q / 2) rest -= widen(out[k]); });
            out[Q / 2] = narrow<real>(rest);
        } else {
            real P = real(0);
            static_for<0, Q / 2>([&](auto K) { constexpr int k = decltype(K)::value; P += (out[k] + out[Q - 1 - k]); });
            out[Q / 2] = Tn - P;
        }
    }
    static_for<0, Q>([&](auto K) {
        constexpr int k = decltype(K)::value, q = q_of(Q, k);
        f[k] = out[k] + real(weight(Q, cls27(q))) * qT;      // + w_i q_T (eq. 27)
    });
    return Tn;
}

// ---- Runge-Kutta stage 1 inside the fused kernel (eqs. 4, 25-26) ------------------------------------
// With kappa_H = kappa_L the term grad kappa . grad T of eq. 4 vanishes and R(T^n) needs nothing beyond what the cell's
// thread already holds: grad T^n and lap T^n (computed for the Marangoni force), u^{n+1}, phi^{n+1}.  The first stage
// then costs one or two stores instead of a kernel that re-reads T^n, phi^{n+1} and u^{n+1} (56-64 B per cell).
// Same expression as rk_stage_march_kernel with dk = 0.
template <typename real>
__device__ __forceinline__ real rk_stage1_local(const StepArgs<real>& A, real phi_new, const real u[3], const real Th[3], real lapT, real qT) {
    const real kap = A.kappa_L + phi_new * A.dkappa;
    const real rcp = (A.rho_L + phi_new * A.drho) * (A.cp_L + phi_new * A.dcp);
    const real adv = u[0] * Th[0] + u[1] * Th[1] + u[2] * Th[2];
    return -adv + (kap * lapT) / rcp + qT;
}

// ---------------------------------------------------------------------------------------------
// fused_step_async_kernel: one thread carries a cell through the whole step.  It first issues ALL of its 27 + 27 + Q_T
// pulls as asynchronous global->shared copies (cp.async, SASS LDGSTS; slot [q][tid], so a thread only
// ever reads what it copied itself and cp.async.wait_group is the only synchronisation needed), then
// does the phi / T stencils, then consumes the three groups in order.  Loads in flight per SM become
// blocks x 128 x (54 + Q_T) x sizeof(real) (187 KB in fp64) instead of whatever the register
// allocator manages to hoist; registers no longer hold prefetched populations.
template <typename real>
__device__ __forceinline__ void cp_async_elem(real* smem_dst, const real* gsrc) {
    const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    if constexpr (sizeof(real) == 8)
        asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(d), "l"(gsrc) : "memory");
    else
        asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(d), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// L2 prefetch for the next wave of blocks (staged kernels).  The block scheduler hands out blocks in index order, so
// the blocks about (resident blocks) ahead of this one start one block lifetime from now.  The blocks of a launch are
// taken in groups of NR = 54 + Q_T + 7 (one per array row the step reads: h, g, f planes, phi and T at z and z + 1,
// u); block r of a group asks L2, with ONE cp.async.bulk.prefetch (SASS UBLKPF.L2) issued by one thread, for row r
// of all NR blocks of the group that lies TCP_PF per cent of a wave ahead (NR x cells_per_block consecutive cells,
// ~70 KB).  The HBM reads of the coming blocks are then in flight while the resident blocks are in their collision
// phase, and their staged copies find the lines in L2: measured 12.4 -> 11.0 ms per step at 400^3 fp64 D3Q7, best at
// half a wave, 40 % for the kernels with two blocks per SM (1.5 waves ahead the lines are evicted again before use and the step
// slows to 14.6 ms).  A hint only: the segment is addressed without the periodic wrap and clamped into the array.
#ifndef TCP_ADDR32
#define TCP_ADDR32 1
#endif

#ifndef TCP_PF
#define TCP_PF 50
#endif
#ifndef TCP_PF2
#define TCP_PF2 40
#endif
template <typename elem, int QT, int AA, int QH = 27, typename Args>
__device__ __forceinline__ void prefetch_next_wave(const Args& A, int cells_per_block, int resident) {
    if constexpr (TCP_PF > 0) {
        if (threadIdx.x != 0) return;
        constexpr int NP = 27 + QH + QT, NR = NP + 7;
        unsigned nsm;
        asm("mov.u32 %0, %%nsmid;" : "=r"(nsm));
        const unsigned r = blockIdx.x % NR;
        const long long N = A.ncell;
        // kernels with two blocks per SM: the optimum is flatter and earlier.  fp64 D3Q19 thermal LB (three blocks, 71 MB of
        // reads + writes in flight per wave): at 50 % some prefetched lines leave L2 before use (46.3 vs 44.4 GB read per launch
        // at 40 %, 13.36 vs 13.26 ms sustained)
        const int pf = (resident == 2 || (sizeof(elem) == 8 && QT == 19 && AA == 0)) ? TCP_PF2 : TCP_PF;
        const long long c0 = (long long)A.cell0 + (long long)(blockIdx.x - r + NR + (pf * resident * nsm) / 100) * cells_per_block;
        if (c0 >= A.cell1) return;
        const elem* base;
        int q27i = 13, plane = 0, Q = 27;
        long long off = c0;
        if (r < 27) { base = A.h_in; plane = q27i = r; }
        else if (r < 27 + QH) {
            base = A.g_in; plane = r - 27; Q = QH;
            static_for<0, QH>([&](auto K) { constexpr int k = decltype(K)::value; if (plane == k) q27i = q_of(QH, k); });
        } else if (r < NP) {
            base = A.f_in; plane = r - 27 - QH; Q = QT;
            static_for<0, QT>([&](auto K) { constexpr int k = decltype(K)::value; if (plane == k) q27i = q_of(QT, k); });
        } else {
            const int j = r - NP;
            if (j < 4) { base = j < 2 ? A.phi_in : A.T_in; if (j & 1) off += (long long)A.nx * A.ny; }
            else { base = A.u; plane = j - 4; }
        }
        if (r < NP) {
            if (AA != 1) off -= cx27(q27i) + A.nx * (cy27(q27i) + (long long)A.ny * cz27(q27i));
            if (AA == 2) plane = Q - 1 - plane;
        }
        long long len = min((long long)NR * cells_per_block, (long long)A.cell1 - c0) + 2;
        off = max(0LL, off);
        len = min(len, N - off);
        if (len <= 0) return;
        const unsigned long long addr = (unsigned long long)__cvta_generic_to_global(base + plane * N + off) & ~15ULL;
        const unsigned bytes = (unsigned)(len * sizeof(elem)) & ~15u;
        if (bytes) asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(addr), "r"(bytes) : "memory");
    }
}

// Residency: (54 + Q_T) x 128 x sizeof(real) bytes of staging per block.  In fp64 three blocks of the
// D3Q15 / D3Q19 variants would take 212-224 KB of the SM's 256 KB, leaving almost no L1 for the
// phi / T stencil loads (measured 0.65 of the HBM peak against 0.81-0.84 for D3Q7 and for D3Q27, which
// only fits two blocks anyway), so those are compiled for two blocks per SM.
// fp64 D3Q15 / D3Q19: h, which is consumed first, is pulled straight into registers together with the stencil loads and
// only g and f are staged (42 / 46 KB per block), so that three blocks fit the shared memory as for D3Q7: 400^3 D3Q15
// 13.25 -> 12.77 ms, D3Q19 13.83 -> 13.39 ms sustained.  D3Q27 (15.16 -> 15.30) keeps h staged.
// D3Q7 has its three blocks anyway and keeps h staged: pulled directly it is 0.6 % faster under the power cap (11.46-11.49 vs
// 11.55 ms) but 3.8 % slower per launch at full clock (ncu 10.77 vs 10.38 ms, DRAM reads 37.5 vs 36.2 GB), as round 1 found.
// The Runge-Kutta paths (Q_T = 0) take it: sustained RK2 10.99-11.02 vs 11.15 ms, +1 % per launch at full clock.
#ifndef TCP_HDIRECT
#define TCP_HDIRECT 1
#endif
// AA in place: round 1 measured a loss of 8-16 %; after the 32-bit offsets, sustained at 400^3: RK2 10.93 vs 11.22 ms, D3Q15 12.96 vs
// 13.12 -- taken; D3Q19 13.84 vs 13.66 and D3Q7 (11.34-11.37 vs 11.46 sustained, but +2.6 % per launch at full clock) -- not taken
template <typename real, int QT, int AA>
__host__ __device__ constexpr bool h_direct() {
    return TCP_HDIRECT && sizeof(real) == 8 && (AA == 0 ? (QT == 0 || QT == 15 || QT == 19) : (QT == 0 || QT == 15));
}

template <typename real, int QT, int AA = 0>
__host__ __device__ constexpr int async_min_blocks() {
    if (sizeof(real) == 4) return 5;   // fp32: 31 KB of staging per block, <= 102 registers; 5 blocks measured +2.7 % over 4
    if (h_direct<real, QT, AA>()) return TCP_MINB;
    return (sizeof(real) == 8 && QT >= 15) ? 2 : TCP_MINB;
}

template <typename real, int QT, bool WALLS, int MODE, int AA, int QH = 27>
__global__ void __launch_bounds__(kBlock, async_min_blocks<real, QT, AA>()) fused_step_async_kernel(const StepArgs<real> A) {
    extern __shared__ __align__(16) unsigned char smem_raw_async[];
    real* stage = reinterpret_cast<real*>(smem_raw_async);     // [27 + QH + QT][kBlock] (27 less if h is not staged)
    const int tid = threadIdx.x;
    const int gtid = A.cell0 + blockIdx.x * kBlock + tid;
    const bool active = gtid < A.cell1;
    const long long N = A.ncell;
    Nbh<WALLS> nb;
    nb.init(A, active ? gtid : A.cell1 - 1);                   // tail lanes shadow the last cell, store nothing
    const int cell = nb.idx;

    // Where the pre-collision population of direction q lives (AA in-place streaming, is a
    // storage permutation only: every step still sees the streamed populations of its cell):
    //   two-grid   : plane q at x - c_q            (wall link: plane opp(q) at x)
    //   AA, even   : plane q at x                  (the odd step / init pushed it there)
    //   AA, odd    : plane opp(q) at x - c_q       (wall link: plane q at x; the even step swapped in place)
    // and where the post-collision one goes:
    //   two-grid   : plane q at x (other grid);  AA even: plane opp(q) at x;
    //   AA odd     : plane q at x + c_q (wall link: plane opp(q) at x, so that the next even step finds it)
    constexpr int aa = AA;   // 0 two-grid, 1 AA even step, 2 AA odd step: compile-time (a run-time switch cost 20 %)
    // Element (plane, off) of a population array as  (base + 9 g N) + (unsigned)((plane - 9 g) N + off),  g = plane / 9: the
    // group base is uniform over the block and the rest fits 32 bits (10 N < 2^32 is validated at creation), so an address
    // is one 32-bit multiply-add and one IMAD.WIDE.U32 instead of a 64-bit (plane N + off) << 3 and a 64-bit add
    // (measured: 4.5 instructions per staged copy before).
    // (the group bases are made opaque to the optimiser, which would otherwise fold 9 g N back into a 64-bit offset)
    const unsigned Nu = (unsigned)A.ncell;
    // fp64 only: the one-cell-per-thread fp32 kernel (odd nx, walls in x) measured 0.5-1 % slower with it
    auto elem = [&](auto* base, int plane, int off) {
        if constexpr (TCP_ADDR32 && sizeof(real) == 8) {
            const int g = plane / 9;
            auto* gb = base + (long long)(9 * g) * N;
            asm("" : "+l"(gb));
            __builtin_assume(__isGlobal(gb));      // the asm hid the address space with the value: keep LDG / STG
            return gb + (unsigned)((unsigned)(plane - 9 * g) * Nu + (unsigned)off);
        } else {
            return base + plane * N + off;
        }
    };
    auto src_of = [&](const real* base, int Q, int k, int q27i) -> const real* {
        const int cx = cx27(q27i), cy = cy27(q27i), cz = cz27(q27i);
        if (aa == 1) return elem(base, k, cell);
        int face = 0;
        const bool bb = WALLS && nb.crossed(-cx, -cy, -cz, face) >= 0;
        if (!WALLS) return elem(base, aa == 2 ? Q - 1 - k : k, nb.at(-cx, -cy, -cz));
        const real* plain = elem(base, aa == 2 ? Q - 1 - k : k, nb.at(-cx, -cy, -cz));
        const real* bounced = elem(base, aa == 2 ? k : Q - 1 - k, cell);
        return bb ? bounced : plain;
    };
    auto dst_of = [&](real* base, int Q, int k, int q27i, bool& wall_link) -> real* {
        const int cx = cx27(q27i), cy = cy27(q27i), cz = cz27(q27i);
        wall_link = false;
        if (aa == 0) return elem(base, k, cell);
        if (aa == 1) return elem(base, Q - 1 - k, cell);
        int face = 0;
        wall_link = WALLS && nb.crossed(cx, cy, cz, face) >= 0;
        return wall_link ? elem(base, Q - 1 - k, cell) : elem(base, k, nb.at(cx, cy, cz));
    };

    real phi_c, G[3], lapPhi, T_c, Th[3], lapT;
    constexpr bool HD = h_direct<real, QT, AA>();
    constexpr int SO = HD ? -27 : 0;                              // slot offset of g and f when h is not staged
    real hd[HD ? 27 : 1];
    if constexpr (HD) {
#pragma unroll
        for (int q = 0; q < 27; ++q) hd[q] = *src_of(A.h_in, 27, q, q);
    } else {
#pragma unroll
        for (int q = 0; q < 27; ++q) cp_async_elem<real>(stage + q * kBlock + tid, src_of(A.h_in, 27, q, q));
    }
    cp_async_commit();
    static_for<0, QH>([&](auto K) {
        constexpr int k = decltype(K)::value, q = q_of(QH, k);
        cp_async_elem<real>(stage + (SO + 27 + k) * kBlock + tid, src_of(A.g_in, QH, k, q));
    });
    cp_async_commit();
    if constexpr (QT > 0) {
        static_for<0, QT>([&](auto K) {
            constexpr int k = decltype(K)::value, q = q_of(QT, k);
            cp_async_elem<real>(stage + (SO + 27 + QH + k) * kBlock + tid, src_of(A.f_in, QT, k, q));
        });
    }
    cp_async_commit();

    // MODE 3 is a roofline calibration, not a step of the method: same pulls, staging and stores, but the
    // stencils and collisions are left out (h, g, f are streamed unchanged; phi, T, u copied through).
    if constexpr (MODE == 3) {
        phi_c = A.phi_in[cell]; T_c = A.T_in[cell];
        G[0] = G[1] = G[2] = Th[0] = Th[1] = Th[2] = lapPhi = lapT = real(0);
    } else {
        stencil27<real, WALLS, false>(A, nb, A.phi_in, phi_c, G, lapPhi);
        stencil27<real, WALLS, true>(A, nb, A.T_in, T_c, Th, lapT);
    }
    real u[3] = {A.u[cell], A.u[N + cell], A.u[2 * N + cell]};

    // (not in the calibration kernel: without arithmetic its blocks are too short-lived, measured 10.98 ms with against 10.5 ms without)
    if constexpr (MODE != 3) prefetch_next_wave<real, QT, AA, QH, StepArgs<real>>(A, kBlock, async_min_blocks<real, QT, AA>());

    real phi_new;
    {
        cp_async_wait<2>();
        real h[27];
#pragma unroll
        for (int q = 0; q < 27; ++q) h[q] = HD ? hd[HD ? q : 0] : stage[q * kBlock + tid];
        if constexpr (MODE == 3) phi_new = phi_c; else phi_new = collide_phase<real, MODE>(A, h, G, phi_c, u);
        if (active) {
#pragma unroll
            for (int q = 0; q < 27; ++q) { bool wl; *dst_of(A.h_out, 27, q, q, wl) = h[q]; }
            A.phi_out[cell] = phi_new;
        }
    }
    {
        cp_async_wait<1>();
        real g[27];
        if constexpr (QH != 27) {
#pragma unroll
            for (int q = 0; q < 27; ++q) g[q] = real(0);     // velocities the hydrodynamic lattice does not have
        }
        static_for<0, QH>([&](auto K) {
            constexpr int k = decltype(K)::value, q = q_of(QH, k);
            g[q] = stage[(SO + 27 + k) * kBlock + tid];
            if (WALLS && aa != 1 && A.moving) g[q] += wall_velocity_term<real, WALLS, QH>(A, nb, q);
        });
        if constexpr (MODE != 3) collide_hydro<real, MODE, QH>(A, g, phi_c, G, lapPhi, T_c, Th, u);
        if (active) {
            static_for<0, QH>([&](auto K) {
                constexpr int k = decltype(K)::value, q = q_of(QH, k);
                bool wl;
                real* dst = dst_of(A.g_out, QH, k, q, wl);
                // AA odd step, link into a moving wall: store what comes back, direction opp(q) with its wall term
                *dst = (WALLS && wl) ? g[q] + wall_velocity_term<real, WALLS, QH>(A, nb, 26 - q) : g[q];
            });
            A.u[cell] = u[0]; A.u[N + cell] = u[1]; A.u[2 * N + cell] = u[2];
        }
    }
    if constexpr (QT == 0 && MODE != 3) {
        if (A.rk1_out && active) {
            const real rhs = rk_stage1_local<real>(A, phi_new, u, Th, lapT, A.q_src ? A.q_src[cell] : real(0));
            A.rk1_out[cell] = T_c + A.rk1_c_out * rhs;
            if (A.rk1_acc) A.rk1_acc[cell] = T_c + A.rk1_c_acc * rhs;
        }
    }
    if constexpr (QT > 0) {
        cp_async_wait<0>();
        real f[QT];
        static_for<0, QT>([&](auto K) {
            constexpr int k = decltype(K)::value, q = q_of(QT, k);
            int face = 0;
            const int ax = aa == 1 ? -1 : nb.crossed(-cx27(q), -cy27(q), -cz27(q), face);
            const real v = stage[(SO + 27 + QH + k) * kBlock + tid];
            if (WALLS && ax >= 0)   // anti-bounce-back (S9): the staged value is f~_opp of the own cell
                f[k] = real(2.0 * weight(QT, cls27(q))) * wall_temperature(A, nb, ax, face, -cx27(q), -cy27(q), -cz27(q)) - v;
            else
                f[k] = v;
        });
        const real qT = A.q_src ? A.q_src[cell] : real(0);
        real Tn;
        if constexpr (MODE == 3) Tn = T_c + qT; else Tn = collide_thermal<real, QT, MODE>(A, f, phi_new, u, qT);
        if (active) {
            static_for<0, QT>([&](auto K) {
                constexpr int k = decltype(K)::value, q = q_of(QT, k);
                bool wl;
                real* dst = dst_of(A.f_out, QT, k, q, wl);
                real v = f[k];
                if (WALLS && wl) {   // AA odd step, link into a wall: store what the next (even) step must read,
                                     // i.e. the anti-bounce-back value -f~_q + 2 w T_w (S9)
                    int face = 0;
                    const int ax = nb.crossed(cx27(q), cy27(q), cz27(q), face);
                    v = real(2.0 * weight(QT, cls27(q))) * wall_temperature(A, nb, ax, face, cx27(q), cy27(q), cz27(q)) - v;
                }
                *dst = v;
            });
            A.T_out[cell] = Tn;
        }
    }
}

// ---------------------------------------------------------------------------------------------
// thermal_only_kernel: the thermal LB update alone, with phi and u frozen (temperature
// pre-initialisation; tcp_relax_temperature).  Same addressing tables as the fused kernel.
template <typename real, bool WALLS, int AA>
__device__ __forceinline__ const real* pop_src(const Nbh<WALLS>& nb, const real* base, long long N, int Q, int k, int q27i) {
    const int cx = cx27(q27i), cy = cy27(q27i), cz = cz27(q27i);
    if (AA == 1) return base + k * N + nb.idx;
    int face = 0;
    const bool bb = WALLS && nb.crossed(-cx, -cy, -cz, face) >= 0;
    const int plane = (bb != (AA == 2)) ? Q - 1 - k : k;
    return base + plane * N + (bb ? nb.idx : nb.at(-cx, -cy, -cz));
}
template <typename real, bool WALLS, int AA>
__device__ __forceinline__ real* pop_dst(const Nbh<WALLS>& nb, real* base, long long N, int Q, int k, int q27i, bool& wall_link) {
    const int cx = cx27(q27i), cy = cy27(q27i), cz = cz27(q27i);
    wall_link = false;
    if (AA == 0) return base + k * N + nb.idx;
    if (AA == 1) return base + (Q - 1 - k) * N + nb.idx;
    int face = 0;
    wall_link = WALLS && nb.crossed(cx, cy, cz, face) >= 0;
    return wall_link ? base + (Q - 1 - k) * N + nb.idx : base + k * N + nb.at(cx, cy, cz);
}

template <typename real, int QT, bool WALLS, int MODE, int AA>
__global__ void __launch_bounds__(kBlock) thermal_only_kernel(const StepArgs<real> A) {
    const int gtid = blockIdx.x * kBlock + threadIdx.x;
    if (gtid >= A.ncell) return;
    const long long N = A.ncell;
    Nbh<WALLS> nb;
    nb.init(A, gtid);
    const int cell = nb.idx;
    real f[QT];
    static_for<0, QT>([&](auto K) {
        constexpr int k = decltype(K)::value, q = q_of(QT, k);
        int face = 0;
        const int ax = AA == 1 ? -1 : nb.crossed(-cx27(q), -cy27(q), -cz27(q), face);
        const real v = *pop_src<real, WALLS, AA>(nb, A.f_in, N, QT, k, q);
        f[k] = (WALLS && ax >= 0) ? real(2.0 * weight(QT, cls27(q))) * wall_temperature(A, nb, ax, face, -cx27(q), -cy27(q), -cz27(q)) - v : v;
    });
    const real u[3] = {A.u[cell], A.u[N + cell], A.u[2 * N + cell]};
    const real qT = A.q_src ? A.q_src[cell] : real(0);
    const real Tn = collide_thermal<real, QT, MODE>(A, f, A.phi_in[cell], u, qT);
    static_for<0, QT>([&](auto K) {
        constexpr int k = decltype(K)::value, q = q_of(QT, k);
        bool wl;
        real* dst = pop_dst<real, WALLS, AA>(nb, A.f_out, N, QT, k, q, wl);
        real v = f[k];
        if (WALLS && wl) {
            int face = 0;
            const int ax = nb.crossed(cx27(q), cy27(q), cz27(q), face);
            v = real(2.0 * weight(QT, cls27(q))) * wall_temperature(A, nb, ax, face, cx27(q), cy27(q), cz27(q)) - v;
        }
        *dst = v;
    });
    A.T_out[cell] = Tn;
}

// ---- AA streaming: a wall temperature that changes while the populations are in the pushed layout -------------
// After tcp_init_fields and after every odd step a link of f~ into a wall is stored already anti-bounced (plane opp(q)
// at the cell, value 2 w T_w - f~_q, see pop_dst), so that the even step that follows needs no boundary code.  The
// stored value carries the T_w of the moment it was written; when tcp_set_wall_temperature replaces the plane of wall
// (axis, face) in that state, the difference 2 w (T_w_new - T_w_old) is folded into the stored links of that wall, and
// the next (even) step then sees exactly what a two-grid pull with the new plane would compute (reading S9).
// One thread per cell of the wall's first fluid layer; `plane_cells` = cells in the tangential plane.
template <typename real, int QT>
__global__ void __launch_bounds__(kBlock) aa_wall_repush_kernel(const StepArgs<real> A, real* __restrict__ f, int axis, int face,
                                                               const real* __restrict__ Tw_new, const real* __restrict__ Tw_old, int plane_cells) {
    const int t = blockIdx.x * kBlock + threadIdx.x;
    if (t >= plane_cells) return;
    const int n[3] = {A.nx, A.ny, A.nz};
    int xyz[3];
    const int a1 = axis == 0 ? 1 : 0, a2 = axis == 2 ? 1 : 2;   // tangential axes, fastest first (plane layout of tcp.h)
    xyz[axis] = face ? n[axis] - 1 : 0;
    xyz[a1] = t % n[a1];
    xyz[a2] = t / n[a1];
    Nbh<true> nb;
    nb.init_xyz(A, xyz[0], xyz[1], xyz[2]);
    const long long N = A.ncell;
    static_for<0, QT>([&](auto K) {
        constexpr int k = decltype(K)::value, q = q_of(QT, k);
        int fc = 0;
        const int ax = nb.crossed(cx27(q), cy27(q), cz27(q), fc);
        if (ax == axis && fc == face) {
            const int i = nb.tangential(axis, cx27(q), cy27(q), cz27(q));
            f[(QT - 1 - k) * N + nb.idx] += real(2.0 * weight(QT, cls27(q))) * (Tw_new[i] - Tw_old[i]);
        }
    });
}

// ---- Runge-Kutta stages of eq. 4 (eqs. 25-26; reading G6) --------------------
template <typename real>
struct RkArgs {
    StepArgs<real> S;        // geometry, walls, phi_in = phi^{n+1}, u = u^{n+1}, q_src
    const real* Y;           // stage field (differentiated)
    const real* Tn;          // T^n
    const real* acc_in;      // RK4 accumulator
    real* out;               // next stage field / T^{n+1}
    real* acc_out;
    real c_out;              // out = Tn + c_out R      (stages 1-3; RK2 stage 2)
    real c_acc;              // acc_out = (first ? Tn : acc_in) + c_acc R
    int mode;                // 0: out only; 1: out and acc from Tn; 2: out and acc from acc_in; 3: out = acc_in + c_acc R
};

// ---- initialisation and read-back --------------------------------------------------------------
template <typename real, int QT, int QH = 27>
__global__ void __launch_bounds__(kBlock) init_kernel(const StepArgs<real> A) {
    const int cell = blockIdx.x * kBlock + threadIdx.x;
    if (cell >= A.ncell) return;
    const long long N = A.ncell;
    const real u[3] = {A.u[cell], A.u[N + cell], A.u[2 * N + cell]};
    const real uu = u[0] * u[0] + u[1] * u[1] + u[2] * u[2];
    // two-grid: population q of the cell goes to plane q at the cell.  AA: the first step is an even one
    // and reads in place, so the equilibria are stored already streamed ("pushed"): plane q at x + c_q,
    // or, for a link into a wall, plane opp(q) at x (for f: as its anti-bounce-back value).
    Nbh<true> nb;
    if (A.aa) {
        const int x = cell % A.nx, t = cell / A.nx;
        nb.init_xyz(A, x, t % A.ny, t / A.ny);
    }
    auto dst_of = [&](real* base, int Q, int k, int q27i, bool& wall_link) -> real* {
        wall_link = false;
        if (!A.aa) return base + k * N + cell;
        int face = 0;
        wall_link = nb.crossed(cx27(q27i), cy27(q27i), cz27(q27i), face) >= 0;
        return wall_link ? base + (Q - 1 - k) * N + cell : base + k * N + nb.at(cx27(q27i), cy27(q27i), cz27(q27i));
    };
    real out[27];
    {
        const real s = A.phi_in[cell];
        const real se = A.eq_sigma * s;
        const real su[3] = {se * u[0], se * u[1], se * u[2]};
        equilibrium_plus_half_force27<real>(se - real(1.5) * se * uu, u, su, su, out);    // eq. 12
        if (A.maxwell) add_product_form27<real, false>(s, u, out);                       // or the Maxwellian
#pragma unroll
        for (int q = 0; q < 27; ++q) { bool wl; *dst_of(A.h_out, 27, q, q, wl) = out[q]; }
    }
    {
        const real sg = A.eq_sigma;
        const real su[3] = {sg * u[0], sg * u[1], sg * u[2]};
        equilibrium_plus_half_force27<real, QH>(-real(1.5) * sg * uu, u, su, su, out);                     // eq. 18, p* = 0
        if (A.maxwell) add_product_form27<real, true>(real(1), u, out);                                   // or w (p* - 1) + Maxwellian
    }
    static_for<0, QH>([&](auto K) {
        constexpr int k = decltype(K)::value, q = q_of(QH, k);
        bool wl;
        real* dst = dst_of(A.g_out, QH, k, q, wl);
        *dst = wl ? out[q] + wall_velocity_term<real, true, QH>(A, nb, 26 - q) : out[q];
    });
    if constexpr (QT > 0) {
        real f[QT];
        thermal_equilibrium<real, QT>(A.T_in[cell], u, f);
        if constexpr (QT == 27) {
            if (A.maxwell) {
#pragma unroll
                for (int q = 0; q < 27; ++q) f[q] = real(0);
                add_product_form27<real, false>(A.T_in[cell], u, f);
            }
        }
        static_for<0, QT>([&](auto K) {
            constexpr int k = decltype(K)::value, q = q_of(QT, k);
            bool wl;
            real* dst = dst_of(A.f_out, QT, k, q, wl);
            real v = f[k];
            if (wl) {
                int face = 0;
                const int ax = nb.crossed(cx27(q), cy27(q), cz27(q), face);
                v = real(2.0 * weight(QT, cls27(q))) * wall_temperature(A, nb, ax, face, cx27(q), cy27(q), cz27(q)) - v;
            }
            *dst = v;
        });
    }
}

// p = c_s^2 rho(phi) sum_q g~_q(x).  pushed = 1: AA layout after init / an odd step, where g~_q(x) sits in
// plane q at x + c_q (plane opp(q) at x for a link into a wall).
template <typename real, int QH = 27>
__global__ void __launch_bounds__(kBlock) pressure_pushed_kernel(const StepArgs<real> A, const real* __restrict__ g, const real* __restrict__ phi,
                                                                real* __restrict__ p) {
    const int cell = blockIdx.x * kBlock + threadIdx.x;
    if (cell >= A.ncell) return;
    const long long N = A.ncell;
    Nbh<true> nb;
    const int x = cell % A.nx, t = cell / A.nx;
    nb.init_xyz(A, x, t % A.ny, t / A.ny);
    real s = real(0);
    static_for<0, QH>([&](auto K) {
        constexpr int k = decltype(K)::value, q = q_of(QH, k);
        int face = 0;
        const bool wl = nb.crossed(cx27(q), cy27(q), cz27(q), face) >= 0;
        s += wl ? g[(QH - 1 - k) * N + cell] : g[k * N + nb.at(cx27(q), cy27(q), cz27(q))];
    });
    p[cell] = real(1.0 / 3.0) * (A.rho_L + phi[cell] * A.drho) * s;
}

template <typename real, int QH = 27>
__global__ void __launch_bounds__(kBlock) pressure_kernel(const real* __restrict__ g, const real* __restrict__ phi, real* __restrict__ p,
                                                         int ncell, real rho_L, real drho) {
    const int cell = blockIdx.x * kBlock + threadIdx.x;
    if (cell >= ncell) return;
    const long long N = ncell;
    real s = real(0);
#pragma unroll
    for (int q = 0; q < QH; ++q) s += g[q * N + cell];
    p[cell] = real(1.0 / 3.0) * (rho_L + phi[cell] * drho) * s;
}

template <typename real>
__global__ void fill_kernel(real* __restrict__ a, long long n, real v) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) a[i] = v;
}

}  // namespace tcp
