// fused_step_pair_kernel: the staged fused step in single precision with TWO x-adjacent cells per thread
// (x even, x + 1) and packed fp32x2 arithmetic (tcp_real.cuh).  A pair costs the instructions of one fp64
// cell: collisions in FFMA2 / FADD2 / FMUL2, one 8-byte store per population plane, 8-byte staged copies
// for the c_x = 0 directions, four loads per stencil row instead of six.  The scalar fp32 kernel spends
// ~2400 instructions per cell on half the bytes and is issue bound at 0.67 of the HBM peak.
//
// Requirements (host-checked, otherwise the scalar kernel runs): x periodic, nx even.  Walls on y / z are
// uniform over a pair; everything else (AA addressing, moving walls, anti-bounce-back, collision modes)
// follows fused_step_async_kernel.
#pragma once
#include "tcp_step.cuh"

namespace tcp {

template <bool WALLS>
struct NbhPair {
    int idx;                 // linear index of the pair's first cell
    int xm1, xp2;            // element offsets of x - 1 and x + 2 from idx (periodic in x)
    int dy[3], dz[3];
    bool lo[3], hi[3];       // y ([1]) and z ([2]) walls touched by the pair's row
    int x, Y[3], Z[3];
    int nx, ny;

    __device__ __forceinline__ void init(const StepArgs<f32x2>& A, int pair) {
        nx = A.nx; ny = A.ny;
        const int hx = A.nx >> 1;
        const int t = (int)fast_div((unsigned)pair, A.div_hx);
        x = 2 * (pair - t * hx);
        const int z = (int)fast_div((unsigned)t, A.div_ny), y = t - z * A.ny;
        const int sy = A.nx, sz = A.nx * A.ny;
        idx = x + sy * y + sz * z;
        xm1 = x > 0 ? -1 : A.nx - 1;
        xp2 = x + 2 < A.nx ? 2 : 2 - A.nx;
        const bool wy = WALLS && A.wall[1], wz = WALLS && A.wall[2];
        dy[1] = dz[1] = 0;
        dy[0] = y > 0 ? -sy : (wy ? 0 : (A.ny - 1) * sy);
        dy[2] = y < A.ny - 1 ? sy : (wy ? 0 : -(A.ny - 1) * sy);
        dz[0] = z > 0 ? -sz : (wz ? 0 : (A.nz - 1) * sz);
        dz[2] = z < A.nz - 1 ? sz : (wz ? 0 : -(A.nz - 1) * sz);
        lo[0] = hi[0] = false;
        lo[1] = wy && y == 0; hi[1] = wy && y == A.ny - 1;
        lo[2] = wz && z == 0; hi[2] = wz && z == A.nz - 1;
        Y[1] = y; Z[1] = z;
        Y[0] = y + dy[0] / sy; Y[2] = y + dy[2] / sy;
        Z[0] = z + dz[0] / sz; Z[2] = z + dz[2] / sz;
    }
    __device__ __forceinline__ int row(int oy, int oz) const { return idx + dy[oy + 1] + dz[oz + 1]; }
    // element offsets of the two cells shifted by ox in {-1, 0, +1} within a row
    __device__ __forceinline__ int first(int ox) const { return ox == 0 ? 0 : (ox < 0 ? xm1 : 1); }
    __device__ __forceinline__ int second(int ox) const { return ox == 0 ? 1 : (ox < 0 ? 0 : xp2); }
    __device__ __forceinline__ int crossed(int oy, int oz, int& face) const {
        if (!WALLS) return -1;
        if (oy == -1 && lo[1]) { face = 0; return 1; }
        if (oy == 1 && hi[1]) { face = 1; return 1; }
        if (oz == -1 && lo[2]) { face = 0; return 2; }
        if (oz == 1 && hi[2]) { face = 1; return 2; }
        return -1;
    }
};

// wall temperatures seen by the two cells shifted by ox, in the ghost row (oy, oz)
template <bool WALLS>
__device__ __forceinline__ f32x2 wall_temperature_pair(const StepArgs<f32x2>& A, const NbhPair<WALLS>& nb, int axis, int face, int ox, int oy, int oz) {
    const int xa = nb.x + nb.first(ox), xb = nb.x + nb.second(ox);
    const int yy = nb.Y[oy + 1], zz = nb.Z[oz + 1];
    const int base = axis == 1 ? zz * nb.nx : yy * nb.nx;
    const float* plane = A.wallT[axis][face];
    return f32x2(plane[base + xa], plane[base + xb]);
}
template <bool WALLS, int QH = 27>
__device__ __forceinline__ f32x2 wall_velocity_term_pair(const StepArgs<f32x2>& A, const NbhPair<WALLS>& nb, int q27i) {
    if (!WALLS || !A.moving) return f32x2(0.0f);
    const int cx = cx27(q27i), cy = cy27(q27i), cz = cz27(q27i);
    int face = 0;
    const int ax = nb.crossed(-cy, -cz, face);
    if (ax < 0) return f32x2(0.0f);
    const float* U = A.wall_u[ax][face];
    return f32x2((float)(6.0 * weight(QH, cls27(q27i))) * ((float)cx * U[0] + (float)cy * U[1] + (float)cz * U[2]));
}

__device__ __forceinline__ void cp_async_4(float* sdst, const float* gsrc) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"((unsigned)__cvta_generic_to_shared(sdst)), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_8(float2* sdst, const float* gsrc) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"((unsigned)__cvta_generic_to_shared(sdst)), "l"(gsrc) : "memory");
}

// 27-point stencil of a pair: per row four values (x-1, x, x+1, x+2); same tensor-product arithmetic as stencil27
template <bool WALLS, bool IS_TEMP>
__device__ __forceinline__ void stencil27_pair(const StepArgs<f32x2>& A, const NbhPair<WALLS>& nb, const float* __restrict__ psi,
                                               f32x2& centre, f32x2 grad[3], f32x2& lap) {
    const f32x2 four(4.0);          // scaling deferred to the end, as in stencil27
    f32x2 SS[3], DSy[3], SDx[3];
#pragma unroll
    for (int oz = -1; oz <= 1; ++oz) {
        f32x2 sx[3], dxv[3];
#pragma unroll
        for (int oy = -1; oy <= 1; ++oy) {
            const float* r = psi + nb.row(oy, oz);
            float v0 = __ldg(r + nb.xm1);
            const float2 mid = __ldg(reinterpret_cast<const float2*>(r));
            float v1 = mid.x, v2 = mid.y;
            float v3 = __ldg(r + nb.xp2);
            if (WALLS && IS_TEMP) {
                int face = 0;
                const int ax = nb.crossed(oy, oz, face);
                if (ax >= 0) {
                    const f32x2 wl = wall_temperature_pair(A, nb, ax, face, -1, oy, oz);   // at x-1, x
                    const f32x2 wr = wall_temperature_pair(A, nb, ax, face, 1, oy, oz);    // at x+1, x+2
                    v0 = 2.0f * wl.v.x - v0; v1 = 2.0f * wl.v.y - v1; v2 = 2.0f * wr.v.x - v2; v3 = 2.0f * wr.v.y - v3;
                }
            }
            if (WALLS && !IS_TEMP && A.wetting) {   // wetting ghost row (reading S20); the row's four values are mirror cells
                int face = 0;
                const int ax = nb.crossed(oy, oz, face);
                if (ax >= 0) {
                    const float a = A.wet_a[ax][face];
                    v0 = wetting_ghost<float>(a, v0); v1 = wetting_ghost<float>(a, v1);
                    v2 = wetting_ghost<float>(a, v2); v3 = wetting_ghost<float>(a, v3);
                }
            }
            const f32x2 m(v0, v1), c(v1, v2), p(v2, v3);
            if (oy == 0 && oz == 0) centre = c;
            sx[oy + 1] = (m + p) + four * c;
            dxv[oy + 1] = p - m;
        }
        SS[oz + 1] = (sx[0] + sx[2]) + four * sx[1];
        DSy[oz + 1] = sx[2] - sx[0];
        SDx[oz + 1] = (dxv[0] + dxv[2]) + four * dxv[1];
    }
    const f32x2 c72(1.0 / 72.0);
    grad[0] = c72 * ((SDx[0] + SDx[2]) + four * SDx[1]);
    grad[1] = c72 * ((DSy[0] + DSy[2]) + four * DSy[1]);
    grad[2] = c72 * (SS[2] - SS[0]);
    lap = f32x2(1.0 / 36.0) * ((SS[0] + SS[2]) + four * SS[1]) - f32x2(6.0) * centre;
}

// Thermal LB, two-grid: h is pulled straight into registers and only g and f are staged; for Q_T >= 15 three blocks then fit
// the shared memory (as in the fp64 D3Q15 / D3Q19 kernels, tcp_step.cuh): 512^3 D3Q15 16.70 -> 16.03 ms, D3Q19 17.29 -> 16.42,
// D3Q27 18.55 -> 18.35, D3Q7 (three blocks either way) 14.34 -> 14.02 sustained; the RK paths (Q_T = 0) lose 0.5-1 % and keep h
// staged
#ifndef TCP_PAIR_ADDR32
#define TCP_PAIR_ADDR32 TCP_ADDR32
#endif
#ifndef TCP_PAIR_HDIRECT
#define TCP_PAIR_HDIRECT 1
#endif
template <int QT, int AA>
__host__ __device__ constexpr bool pair_h_direct() { return TCP_PAIR_HDIRECT && QT > 0 && AA == 0; }
template <int QT, int AA = 0>
__host__ __device__ constexpr int pair_min_blocks() { return (QT >= 15 && !pair_h_direct<QT, AA>()) ? 2 : TCP_MINB; }

template <int QT, bool WALLS, int MODE, int AA, int QH = 27>
__global__ void __launch_bounds__(kBlock, pair_min_blocks<QT, AA>()) fused_step_pair_kernel(const StepArgs<f32x2> A) {
    using real = f32x2;
    extern __shared__ __align__(16) unsigned char smem_raw_pair[];
    float2* stage = reinterpret_cast<float2*>(smem_raw_pair) + threadIdx.x;     // [54 + QT][kBlock], this thread's column
    const int npairs = A.cell1 >> 1;                        // cell0, cell1 are even (whole rows of an even nx)
    const int gp = (A.cell0 >> 1) + blockIdx.x * kBlock + threadIdx.x;
    const bool active = gp < npairs;
    const long long N = A.ncell;
    NbhPair<WALLS> nb;
    nb.init(A, active ? gp : npairs - 1);
    const int cell = nb.idx;
    constexpr int aa = AA;

    // element (plane, off) of a population array with a 32-bit offset from the uniform base of its group of 9 planes
    // (fused_step_async_kernel, tcp_step.cuh)
    const unsigned Nu = (unsigned)A.ncell;
    // (only where h is staged too: with h pulled into registers the variants lose -- 512^3 sustained D3Q7 13.48 vs 12.67 ms,
    // D3Q19 15.88 vs 15.30, more spills -- while RK2 gains, 12.10 vs 12.46-12.50, and AA is unchanged)
    constexpr bool A32 = TCP_PAIR_ADDR32 && !pair_h_direct<QT, AA>();
    auto elem = [&](auto* base, int plane, int off) {
        if constexpr (A32) {
            const int g = plane / 9;
            auto* gb = base + (long long)(9 * g) * N;
            asm("" : "+l"(gb));
            __builtin_assume(__isGlobal(gb));
            return gb + (unsigned)((unsigned)(plane - 9 * g) * Nu + (unsigned)off);
        } else {
            return base + plane * N + off;
        }
    };
    // issue the pulls of both cells of direction (Q, k, q27) into the slot (addressing table: fused_step_async_kernel)
    auto issue = [&](float2* slot, const float* base, int Q, int k, int q27i) {
        const int cx = cx27(q27i), cy = cy27(q27i), cz = cz27(q27i);
        if (aa == 1) { cp_async_8(slot, elem(base, k, cell)); return; }
        int face = 0;
        const bool bb = WALLS && nb.crossed(-cy, -cz, face) >= 0;
        const int plane = (bb != (aa == 2)) ? Q - 1 - k : k;
        if (bb) { cp_async_8(slot, elem(base, plane, cell)); return; }
        const float* r = elem(base, plane, nb.row(-cy, -cz));
        if (cx == 0) cp_async_8(slot, r);
        else {
            cp_async_4(reinterpret_cast<float*>(slot), r + nb.first(-cx));
            cp_async_4(reinterpret_cast<float*>(slot) + 1, r + nb.second(-cx));
        }
    };
    // store the post-collision pair of direction (Q, k, q27); returns through wall_link whether it went into a wall
    auto put = [&](float* base, int Q, int k, int q27i, real v, bool& wall_link) {
        const int cx = cx27(q27i), cy = cy27(q27i), cz = cz27(q27i);
        wall_link = false;
        if (aa == 0) { *reinterpret_cast<float2*>(elem(base, k, cell)) = v.v; return; }
        if (aa == 1) { *reinterpret_cast<float2*>(elem(base, Q - 1 - k, cell)) = v.v; return; }
        int face = 0;
        wall_link = WALLS && nb.crossed(cy, cz, face) >= 0;
        if (wall_link) { *reinterpret_cast<float2*>(elem(base, Q - 1 - k, cell)) = v.v; return; }
        float* r = elem(base, k, nb.row(cy, cz));
        if (cx == 0) *reinterpret_cast<float2*>(r) = v.v;
        else { r[nb.first(cx)] = v.v.x; r[nb.second(cx)] = v.v.y; }
    };

    // the same addressing with plain loads (pair_h_direct)
    auto fetch = [&](const float* base, int Q, int k, int q27i) -> float2 {
        const int cx = cx27(q27i), cy = cy27(q27i), cz = cz27(q27i);
        if (aa == 1) return *reinterpret_cast<const float2*>(elem(base, k, cell));
        int face = 0;
        const bool bb = WALLS && nb.crossed(-cy, -cz, face) >= 0;
        const int plane = (bb != (aa == 2)) ? Q - 1 - k : k;
        if (bb) return *reinterpret_cast<const float2*>(elem(base, plane, cell));
        const float* r = elem(base, plane, nb.row(-cy, -cz));
        if (cx == 0) return *reinterpret_cast<const float2*>(r);
        return make_float2(r[nb.first(-cx)], r[nb.second(-cx)]);
    };
    constexpr bool HD = pair_h_direct<QT, AA>();
    constexpr int SO = HD ? -27 : 0;
    // The phi / T stencil loads and u.  With the D3Q7 thermal LB (two-grid) they are issued BEFORE the staged copies of g and f:
    // the LSU works through its queue in order, the stencils and h are what the thread needs first, and 34 cp.async of 8 LSU
    // cycles each would otherwise sit in front of them.  Measured sustained at 512^3: D3Q7 12.58-12.60 vs 13.00-13.05 ms; the
    // other variants lose 1-2 % that way (RK2 12.51-12.53 vs 12.39-12.44, AA 13.68-13.71 vs 13.42-13.44, D3Q19 unchanged)
    // and keep the stencils last; so does the fp64 kernel (D3Q7 11.98-12.00 vs 12.02-12.06, RK2 11.71-11.74 vs 11.34-11.38).
    constexpr bool SF = QT == 7 && AA == 0;
    real phi_c, G[3], lapPhi, T_c, Th[3], lapT, u[3];
    auto load_fields = [&]() {
        stencil27_pair<WALLS, false>(A, nb, A.phi_in, phi_c, G, lapPhi);
        stencil27_pair<WALLS, true>(A, nb, A.T_in, T_c, Th, lapT);
#pragma unroll
        for (int al = 0; al < 3; ++al) { const float2 t = *reinterpret_cast<const float2*>(A.u + al * N + cell); u[al] = real(t.x, t.y); }
    };
    float2 hd[HD ? 27 : 1];
    if constexpr (HD) {
#pragma unroll
        for (int q = 0; q < 27; ++q) hd[q] = fetch(A.h_in, 27, q, q);
    } else {
#pragma unroll
        for (int q = 0; q < 27; ++q) issue(stage + q * kBlock, A.h_in, 27, q, q);
    }
    cp_async_commit();
    if constexpr (SF) load_fields();
    static_for<0, QH>([&](auto K) { constexpr int k = decltype(K)::value; issue(stage + (SO + 27 + k) * kBlock, A.g_in, QH, k, q_of(QH, k)); });
    cp_async_commit();
    if constexpr (QT > 0)
        static_for<0, QT>([&](auto K) { constexpr int k = decltype(K)::value; issue(stage + (SO + 27 + QH + k) * kBlock, A.f_in, QT, k, q_of(QT, k)); });
    cp_async_commit();

    if constexpr (!SF) load_fields();

    prefetch_next_wave<float, QT, AA, QH, StepArgs<f32x2>>(A, 2 * kBlock, pair_min_blocks<QT, AA>());

    real phi_new;
    {
        cp_async_wait<2>();
        real h[27];
#pragma unroll
        for (int q = 0; q < 27; ++q) h[q].v = HD ? hd[HD ? q : 0] : stage[q * kBlock];
        phi_new = collide_phase<real, MODE>(A, h, G, phi_c, u);
        if (active) {
#pragma unroll
            for (int q = 0; q < 27; ++q) { bool wl; put(A.h_out, 27, q, q, h[q], wl); }
            *reinterpret_cast<float2*>(A.phi_out + cell) = phi_new.v;
        }
    }
    {
        cp_async_wait<1>();
        real g[27];
        if constexpr (QH != 27) {
#pragma unroll
            for (int q = 0; q < 27; ++q) g[q] = real(0.0f);   // velocities the hydrodynamic lattice does not have
        }
        static_for<0, QH>([&](auto K) {
            constexpr int k = decltype(K)::value, q = q_of(QH, k);
            g[q].v = stage[(SO + 27 + k) * kBlock];
            if (WALLS && aa != 1 && A.moving) g[q] += wall_velocity_term_pair<WALLS, QH>(A, nb, q);
        });
        collide_hydro<real, MODE, QH>(A, g, phi_c, G, lapPhi, T_c, Th, u);
        if (active) {
            static_for<0, QH>([&](auto K) {
                constexpr int k = decltype(K)::value, q = q_of(QH, k);
                // AA odd step, link into a moving wall: what comes back is direction opp(q) with its wall term
                int face = 0;
                const bool into_wall = WALLS && aa == 2 && nb.crossed(cy27(q), cz27(q), face) >= 0;
                bool wl;
                put(A.g_out, QH, k, q, into_wall ? g[q] + wall_velocity_term_pair<WALLS, QH>(A, nb, 26 - q) : g[q], wl);
            });
#pragma unroll
            for (int al = 0; al < 3; ++al) *reinterpret_cast<float2*>(A.u + al * N + cell) = u[al].v;
        }
    }
    if constexpr (QT == 0) {
        if (A.rk1_out && active) {   // Runge-Kutta stage 1 of both cells (rk_stage1_local, tcp_step.cuh)
            real qT(0.0f);
            if (A.q_src) { const float2 t = *reinterpret_cast<const float2*>(A.q_src + cell); qT = real(t.x, t.y); }
            const real rhs = rk_stage1_local<real>(A, phi_new, u, Th, lapT, qT);
            *reinterpret_cast<float2*>(A.rk1_out + cell) = (T_c + A.rk1_c_out * rhs).v;
            if (A.rk1_acc) *reinterpret_cast<float2*>(A.rk1_acc + cell) = (T_c + A.rk1_c_acc * rhs).v;
        }
    }
    if constexpr (QT > 0) {
        cp_async_wait<0>();
        real f[QT];
        static_for<0, QT>([&](auto K) {
            constexpr int k = decltype(K)::value, q = q_of(QT, k);
            int face = 0;
            const int ax = aa == 1 ? -1 : nb.crossed(-cy27(q), -cz27(q), face);
            real v; v.v = stage[(SO + 27 + QH + k) * kBlock];
            if (WALLS && ax >= 0)   // anti-bounce-back (S9): T_w at the tangential position of each lane's source cell
                v = real(2.0 * weight(QT, cls27(q))) * wall_temperature_pair(A, nb, ax, face, -cx27(q), -cy27(q), -cz27(q)) - v;
            f[k] = v;
        });
        real qT(0.0f);
        if (A.q_src) { const float2 t = *reinterpret_cast<const float2*>(A.q_src + cell); qT = real(t.x, t.y); }
        const real Tn = collide_thermal<real, QT, MODE>(A, f, phi_new, u, qT);
        if (active) {
            static_for<0, QT>([&](auto K) {
                constexpr int k = decltype(K)::value, q = q_of(QT, k);
                real v = f[k];
                int face = 0;
                const int ax = (WALLS && aa == 2) ? nb.crossed(cy27(q), cz27(q), face) : -1;
                if (ax >= 0)   // AA odd step, link into a wall: store its anti-bounce-back value (S9)
                    v = real(2.0 * weight(QT, cls27(q))) * wall_temperature_pair(A, nb, ax, face, cx27(q), cy27(q), cz27(q)) - v;
                bool wl;
                put(A.f_out, QT, k, q, v, wl);
            });
            *reinterpret_cast<float2*>(A.T_out + cell) = Tn.v;
        }
    }
}

}  // namespace tcp
