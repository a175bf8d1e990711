// Kernels of the coupled step.
//
//   fused_step_kernel   one pass per time step: phase-field LB (eqs. 10-15), hydrodynamic LB
//                       (eqs. 16-22 with the forces of eqs. 7-9) and, for QT > 0, the thermal LB
//                       (eqs. 27-29).  All three read only time level n outside their own cell
//                       (reading S16), so one thread carries a cell through all of
//                       them and the phi / T halos are read once.
//   rk_stage_kernel     one Runge-Kutta stage of eq. 4 (eqs. 25-26)
//   init_kernel         populations <- equilibria
//   pressure_kernel     p = c_s^2 rho(phi) sum g~
#pragma once
#include <type_traits>
#include <utility>

#include "tcp_device.cuh"

namespace tcp {


// ---------------------------------------------------------------------------------------------
// thermal lattice helpers (stencil Q, compact index k)

// out_k = s w_k [1 + 3 c.u + 4.5 (c.u)^2 - 1.5 u.u]   (eq. 12 with phi -> T)
template <typename real, int Q>
__device__ __forceinline__ void thermal_equilibrium(real s, const real u[3], real out[Q]) {
    const real base = real(1) - real(1.5) * (u[0] * u[0] + u[1] * u[1] + u[2] * u[2]);
    static_for<0, Q>([&](auto K) {
        constexpr int k = decltype(K)::value, q = q_of(Q, k);
        constexpr int cx = cx27(q), cy = cy27(q), cz = cz27(q);
        constexpr double w = weight(Q, cls27(q));
        const real cu = real(cx) * u[0] + real(cy) * u[1] + real(cz) * u[2];
        out[k] = s * real(w) * (base + cu * (real(3) + real(4.5) * cu));
    });
}

// out_k += populations with first-order central moments m, all other basis central moments 0.
// Their raw moments are M_b = (m . grad) b (u) for every basis function b of reading S2; the
// populations follow from the stencil's raw-moment inversion.
template <typename real, int Q>
__device__ __forceinline__ void add_first_order_thermal(const real m[3], const real u[3], real out[Q]) {
    static_assert(Q == 7 || Q == 15 || Q == 19, "D3Q27 uses add_first_order27");
    const real M2[3] = {real(2) * u[0] * m[0], real(2) * u[1] * m[1], real(2) * u[2] * m[2]};
    const real sumM2 = M2[0] + M2[1] + M2[2];
    if constexpr (Q == 7) {
        static_for<0, Q>([&](auto K) {
            constexpr int k = decltype(K)::value, q = q_of(Q, k);
            constexpr int c[3] = {cx27(q), cy27(q), cz27(q)};
            if constexpr (cls27(q) == 0) {
                out[k] += -sumM2;
            } else {
                constexpr int a = c[0] != 0 ? 0 : (c[1] != 0 ? 1 : 2);
                out[k] += real(0.5) * (M2[a] + real(c[a]) * m[a]);
            }
        });
    } else if constexpr (Q == 19) {
        // pair (a,b): m22 = d(x_a^2 x_b^2), m12 = d(x_a x_b^2), m21 = d(x_a^2 x_b), m11 = d(x_a x_b)
        real m22[3], m12[3], m21[3], m11[3];   // pair index p: 0 = (x,y), 1 = (x,z), 2 = (y,z)
        static_for<0, 3>([&](auto Pp) {
            constexpr int p = decltype(Pp)::value, a = (p == 2 ? 1 : 0), b = (p == 0 ? 1 : 2);
            m22[p] = real(2) * u[a] * u[b] * (u[b] * m[a] + u[a] * m[b]);
            m12[p] = u[b] * u[b] * m[a] + real(2) * u[a] * u[b] * m[b];
            m21[p] = real(2) * u[a] * u[b] * m[a] + u[a] * u[a] * m[b];
            m11[p] = m[a] * u[b] + m[b] * u[a];
        });
        static_for<0, Q>([&](auto K) {
            constexpr int k = decltype(K)::value, q = q_of(Q, k);
            constexpr int c[3] = {cx27(q), cy27(q), cz27(q)};
            if constexpr (cls27(q) == 0) {
                out[k] += -sumM2 + (m22[0] + m22[1] + m22[2]);
            } else if constexpr (cls27(q) == 1) {
                constexpr int a = c[0] != 0 ? 0 : (c[1] != 0 ? 1 : 2);
                // pairs containing axis a, and the moment of x_a x_other^2 in each
                constexpr int p1 = (a == 0 ? 0 : (a == 1 ? 0 : 1));
                constexpr int p2 = (a == 0 ? 1 : (a == 1 ? 2 : 2));
                const real q1 = (a == 0) ? m12[0] : (a == 1 ? m21[0] : m21[1]);
                const real q2 = (a == 0) ? m12[1] : (a == 1 ? m12[2] : m21[2]);
                out[k] += real(0.5) * ((M2[a] - m22[p1] - m22[p2]) + real(c[a]) * (m[a] - q1 - q2));
            } else {
                constexpr int p = (c[2] == 0 ? 0 : (c[1] == 0 ? 1 : 2));
                constexpr int a = (p == 2 ? 1 : 0), b = (p == 0 ? 1 : 2);
                out[k] += real(0.25) * (m22[p] + real(c[a]) * m12[p] + real(c[b]) * m21[p] + real(c[a] * c[b]) * m11[p]);
            }
        });
    } else {   // Q == 15
        const real ux = u[0], uy = u[1], uz = u[2], mx = m[0], my = m[1], mz = m[2];
        const real Mxy = mx * uy + my * ux, Mxz = mx * uz + mz * ux, Myz = my * uz + mz * uy;
        const real Mxyz = mx * uy * uz + my * ux * uz + mz * ux * uy;
        const real A3[3] = {mx * (uy * uy + uz * uz) + real(2) * ux * (uy * my + uz * mz),
                            my * (ux * ux + uz * uz) + real(2) * uy * (ux * mx + uz * mz),
                            mz * (ux * ux + uy * uy) + real(2) * uz * (ux * mx + uy * my)};
        const real m4 = real(2) * (ux * mx * (uy * uy + uz * uz) + uy * my * (ux * ux + uz * uz) + uz * mz * (ux * ux + uy * uy));
        const real C = m4 * real(1.0 / 3.0);
        static_for<0, Q>([&](auto K) {
            constexpr int k = decltype(K)::value, q = q_of(Q, k);
            constexpr int c[3] = {cx27(q), cy27(q), cz27(q)};
            if constexpr (cls27(q) == 0) {
                out[k] += -sumM2 + real(2) * C;
            } else if constexpr (cls27(q) == 1) {
                constexpr int a = c[0] != 0 ? 0 : (c[1] != 0 ? 1 : 2);
                out[k] += real(0.5) * ((M2[a] - C) + real(c[a]) * (m[a] - real(0.5) * A3[a]));
            } else {
                out[k] += real(0.125) * (C + real(0.5) * (real(c[0]) * A3[0] + real(c[1]) * A3[1] + real(c[2]) * A3[2])
                                         + real(c[0] * c[1]) * Mxy + real(c[0] * c[2]) * Mxz + real(c[1] * c[2]) * Myz
                                         + real(c[0] * c[1] * c[2]) * Mxyz);
            }
        });
    }
}

}  // namespace tcp
