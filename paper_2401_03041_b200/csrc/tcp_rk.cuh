// rk_stage_march_kernel: one Runge-Kutta stage of eq. 4 (eqs. 25-26) as a z-marching stencil kernel.
//
// The stage needs the 27-point gradient and Laplacian of the stage field Y and the gradient of
// phi^{n+1} and moves only 7-9 values per cell, so 54 global (or shared) loads per cell would make it
// load-issue bound far above its HBM floor (measured: 1.8 ms per stage at 400^3 against 0.55 ms).
// Here a block owns a TX x TY tile in (x, y) and walks a chunk of z planes: each plane's tile + halo
// is staged once in shared memory (ghost rules applied by the loader), every thread reduces its 3 x 3
// in-plane neighbourhood to S_xS_y, D_xS_y, S_xD_y (9 shared loads per field and plane) and keeps
// those for three consecutive planes in registers; the z-direction of the tensor-product stencil
// (reading S3) then closes on registers.  Same arithmetic, in the same order, as stencil27.
#pragma once
#include "tcp_step.cuh"

namespace tcp {

// fp64 without the phi tile: three blocks per SM (80 registers, 20-64 B of spills) measured 1 % faster on RK4 than two
#ifndef TCP_RK_RING
#define TCP_RK_RING 3
#endif
#ifndef TCP_RK_B3
#define TCP_RK_B3 1
#endif
constexpr int kRkTX = 32, kRkTY = 8, kRkCZ = 32;   // chunks of 16-100 planes: within 1 %
// Residency: with the cell data requested one plane ahead the fp64 kernel needs
// 119 registers -> 2 blocks of 256 per SM without spills (3 blocks: 80-116 B of spills and 8-15 % slower);
// the fp32 kernel fits 3 blocks.
template <typename real, bool HAS_DK>
constexpr int rk_min_blocks() { return sizeof(real) == 8 && (HAS_DK || !TCP_RK_B3) ? 2 : 3; }

// bytes of the cell-data ring of rk_stage_march_kernel (dynamic shared memory): TCP_RK_RING planes x 7 values x the tile
template <typename real>
constexpr size_t rk_ring_bytes() { return (size_t)TCP_RK_RING * 7 * kRkTX * kRkTY * sizeof(real); }

template <typename real>
struct Plane3 {          // in-plane reductions of one field on one z plane
    real S, Dx, Dy, c;
};

// MODE = RkArgs::mode and HAS_Q = (q_src != nullptr) are compile-time here, and the plane loop is unrolled three
// times so that the three-plane register window (z-1, z, z+1) rotates by renaming instead of by moves: 273 -> 2xx
// instructions per cell (ncu: the kernel keeps the issue slots 54 % busy, so instructions are what it is made of).
// HAS_DK = (kappa_H != kappa_L): with equal conductivities grad kappa . grad T of eq. 4 vanishes identically, so the
// phi tile, its nine shared loads and its reductions are left out and phi is read at the cell only (for rho c_p).
template <typename real, bool WALLS, int MODE, bool HAS_Q, bool HAS_DK>
__global__ void __launch_bounds__(kRkTX * kRkTY, rk_min_blocks<real, HAS_DK>()) rk_stage_march_kernel(const RkArgs<real> R) {
    const StepArgs<real>& A = R.S;
    constexpr int TX = kRkTX, TY = kRkTY, PX = TX + 2, PY = TY + 2, PE = PX * PY;
    __shared__ real tileY[2][PE], tileP[2][PE];
    const int tid = threadIdx.y * TX + threadIdx.x;
    // planes [cell0, cell1) / (nx ny): the whole box, or the boundary planes / the interior of a slab
    const int zfirst = A.cell0 / (A.nx * A.ny), zend = A.cell1 / (A.nx * A.ny);
    const int bx0 = blockIdx.x * TX, by0 = blockIdx.y * TY, z0 = zfirst + blockIdx.z * kRkCZ;
    const int nzc = min(kRkCZ, zend - z0);
    const int x = bx0 + threadIdx.x, y = by0 + threadIdx.y;
    const bool inside = x < A.nx && y < A.ny;
    const long long N = A.ncell;
    const int sy = A.nx, sz = A.nx * A.ny;
    const bool wx = WALLS && A.wall[0], wy = WALLS && A.wall[1], wz = WALLS && A.wall[2];

    // loader.  Thread t owns halo-tile elements e = t and t + TX*TY (if < PE); their in-plane source
    // coordinates and wall flags do not depend on z, so they are resolved once.
    constexpr int NE = (PE + TX * TY - 1) / (TX * TY);
    int e_idx2d[NE], e_tang_x[NE], e_tang_y[NE], e_fx[NE], e_fy[NE];
    bool e_on[NE];
#pragma unroll
    for (int i = 0; i < NE; ++i) {
        const int e = tid + i * TX * TY;
        e_on[i] = e < PE;
        const int ty = e / PX, tx = e - ty * PX;
        int X = bx0 + tx - 1, Y = by0 + ty - 1, fx = -1, fy = -1;
        if (X < 0) { if (wx) { fx = 0; X = 0; } else X += A.nx; }
        else if (X >= A.nx) { if (X == A.nx) { if (wx) { fx = 1; X = A.nx - 1; } else X = 0; } else X = A.nx - 1; }
        if (Y < 0) { if (wy) { fy = 0; Y = 0; } else Y += A.ny; }
        else if (Y >= A.ny) { if (Y == A.ny) { if (wy) { fy = 1; Y = A.ny - 1; } else Y = 0; } else Y = A.ny - 1; }
        if (X < 0) X = 0;          // nx == 1 corner of an overhanging tile
        if (Y < 0) Y = 0;
        e_idx2d[i] = X + sy * Y; e_fx[i] = fx; e_fy[i] = fy; e_tang_x[i] = X; e_tang_y[i] = Y;
    }
    real pfY[NE], pfP[NE];          // prefetched plane (in flight while the previous one is consumed)
    auto fetch_plane = [&](int zreq) {
        int fz = -1, Z = zreq;
        if (Z < 0) { if (wz) { fz = 0; Z = 0; } else Z += A.nz; }
        else if (Z >= A.nz) { if (wz) { fz = 1; Z = A.nz - 1; } else Z -= A.nz; }
#pragma unroll
        for (int i = 0; i < NE; ++i) {
            if (!e_on[i]) continue;
            const int idx = e_idx2d[i] + sz * Z;
            real vy = __ldg(R.Y + idx);
            if (HAS_DK) {
                real vp = __ldg(A.phi_in + idx);
                if (WALLS && A.wetting) {   // wetting ghost (reading S20): first crossed wall in x, y, z order, as in stencil27
                    if (e_fx[i] >= 0) vp = wetting_ghost<real>(A.wet_a[0][e_fx[i]], vp);
                    else if (e_fy[i] >= 0) vp = wetting_ghost<real>(A.wet_a[1][e_fy[i]], vp);
                    else if (fz >= 0) vp = wetting_ghost<real>(A.wet_a[2][fz], vp);
                }
                pfP[i] = vp;
            }
            if (WALLS) {   // Dirichlet ghost 2 T_w - Y(mirror); first crossed axis in x, y, z order (S9, S17)
                if (e_fx[i] >= 0) vy = real(2) * A.wallT[0][e_fx[i]][Z * A.ny + e_tang_y[i]] - vy;
                else if (e_fy[i] >= 0) vy = real(2) * A.wallT[1][e_fy[i]][Z * A.nx + e_tang_x[i]] - vy;
                else if (fz >= 0) vy = real(2) * A.wallT[2][fz][e_tang_y[i] * A.nx + e_tang_x[i]] - vy;
            }
            pfY[i] = vy;
        }
    };
    auto store_plane = [&](int buf) {
#pragma unroll
        for (int i = 0; i < NE; ++i)
            if (e_on[i]) { tileY[buf][tid + i * TX * TY] = pfY[i]; if (HAS_DK) tileP[buf][tid + i * TX * TY] = pfP[i]; }
    };
    const real four = real(4), c72 = real(1.0 / 72.0), c36 = real(1.0 / 36.0);   // scaling deferred to the end, as in stencil27
    auto reduce_plane = [&](const real* t) {
        Plane3<real> P;
        real sx[3], dxv[3];
#pragma unroll
        for (int oy = 0; oy < 3; ++oy) {
            const real* row = t + (threadIdx.y + oy) * PX + threadIdx.x;
            const real m = row[0], c = row[1], p = row[2];
            if (oy == 1) P.c = c;
            sx[oy] = (m + p) + four * c;
            dxv[oy] = p - m;
        }
        P.S = (sx[0] + sx[2]) + four * sx[1];
        P.Dy = sx[2] - sx[0];
        P.Dx = (dxv[0] + dxv[2]) + four * dxv[1];
        return P;
    };

    // plane p_j = z0 - 1 + j lives in buffer j & 1
    Plane3<real> Ym, Yc, Yp, Pm, Pc, Pp;   // planes z-1, z, z+1 of Y and phi
    fetch_plane(z0 - 1); store_plane(0);
    fetch_plane(z0); store_plane(1);
    fetch_plane(z0 + 1);                   // stays in registers until iteration 0 stores it
    __syncthreads();
    Ym = reduce_plane(tileY[0]); Yc = reduce_plane(tileY[1]);
    if (HAS_DK) { Pm = reduce_plane(tileP[0]); Pc = reduce_plane(tileP[1]); }
    __syncthreads();                       // buffer 0 may now be overwritten
    // cell data (u, T^n, accumulator, source, phi) of plane z0 + k: every thread copies its own cell's values D - 1 planes
    // ahead (RK4 -1.5 % against one plane ahead in registers) with cp.async into its slot of a shared-memory ring (it reads only what it copied itself, so
    // cp.async.wait_group is all the synchronisation this needs); no registers are held while they are in flight
    constexpr int D = TCP_RK_RING, NV = 7, RING = NV * TX * TY;
    extern __shared__ __align__(16) unsigned char rk_ring_raw[];
    real* ring = reinterpret_cast<real*>(rk_ring_raw);
    auto request_cell = [&](int k) {          // plane z0 + k -> ring slot k % D
        if (inside && k < nzc) {
            const int c = x + sy * y + sz * (z0 + k);
            real* slot = ring + (k % D) * RING + tid;
            cp_async_elem<real>(slot, A.u + c);
            cp_async_elem<real>(slot + TX * TY, A.u + N + c);
            cp_async_elem<real>(slot + 2 * TX * TY, A.u + 2 * N + c);
            if (MODE != 3) cp_async_elem<real>(slot + 3 * TX * TY, R.Tn + c);
            if (MODE >= 2) cp_async_elem<real>(slot + 4 * TX * TY, R.acc_in + c);
            if (HAS_Q) cp_async_elem<real>(slot + 5 * TX * TY, A.q_src + c);
            if (!HAS_DK) cp_async_elem<real>(slot + 6 * TX * TY, A.phi_in + c);
        }
        cp_async_commit();                    // one group per plane, empty or not: the wait below counts groups
    };
#pragma unroll
    for (int j = 0; j < D - 1; ++j) request_cell(j);
    const real c_out = R.c_out, c_acc = R.c_acc;
    // one plane: (Ym, Yc) and (Pm, Pc) hold planes z-1, z; Yp / Pp receive plane z+1
    auto plane = [&](int k, const Plane3<real>& Ym, const Plane3<real>& Yc, Plane3<real>& Yp,
                     const Plane3<real>& Pm, const Plane3<real>& Pc, Plane3<real>& Pp) {
        const int buf = k & 1;
        const int cell = x + sy * y + sz * (z0 + k);
        request_cell(k + D - 1);
        cp_async_wait<D - 1>();                    // plane k's group has landed
        const real* slot = ring + (k % D) * RING + tid;
        real u[3] = {real(0), real(0), real(0)}, Tn = real(0), acc = real(0), qT = real(0), phi_here = real(0);
        if (inside) {
            u[0] = slot[0]; u[1] = slot[TX * TY]; u[2] = slot[2 * TX * TY];
            if (MODE != 3) Tn = slot[3 * TX * TY];
            if (MODE >= 2) acc = slot[4 * TX * TY];
            if (HAS_Q) qT = slot[5 * TX * TY];
            if (!HAS_DK) phi_here = slot[6 * TX * TY];
        }
        store_plane(buf);                          // plane z0 + k + 1
        if (k + 1 < nzc) fetch_plane(z0 + k + 2);  // next one: its latency hides behind this iteration
        __syncthreads();
        Yp = reduce_plane(tileY[buf]);
        if (HAS_DK) Pp = reduce_plane(tileP[buf]);
        if (inside) {
            real gY[3], G[3] = {real(0), real(0), real(0)};
            gY[0] = c72 * ((Ym.Dx + Yp.Dx) + four * Yc.Dx);
            gY[1] = c72 * ((Ym.Dy + Yp.Dy) + four * Yc.Dy);
            gY[2] = c72 * (Yp.S - Ym.S);
            const real lapY = c36 * ((Ym.S + Yp.S) + four * Yc.S) - real(6) * Yc.c;
            if (HAS_DK) {
                G[0] = c72 * ((Pm.Dx + Pp.Dx) + four * Pc.Dx);
                G[1] = c72 * ((Pm.Dy + Pp.Dy) + four * Pc.Dy);
                G[2] = c72 * (Pp.S - Pm.S);
            }
            const real phi_c = HAS_DK ? Pc.c : phi_here;
            const real kap = A.kappa_L + phi_c * A.dkappa;
            const real rcp = (A.rho_L + phi_c * A.drho) * (A.cp_L + phi_c * A.dcp);
            const real adv = u[0] * gY[0] + u[1] * gY[1] + u[2] * gY[2];
            const real dk = HAS_DK ? A.dkappa * (G[0] * gY[0] + G[1] * gY[1] + G[2] * gY[2]) : real(0);
            const real rhs = -adv + (dk + kap * lapY) / rcp + qT;
            if (MODE == 3) {
                R.out[cell] = acc + c_acc * rhs;
            } else {
                R.out[cell] = Tn + c_out * rhs;
                if (MODE == 1) R.acc_out[cell] = Tn + c_acc * rhs;
                if (MODE == 2) R.acc_out[cell] = acc + c_acc * rhs;
            }
        }
        // no second barrier: iteration k+1 overwrites the OTHER buffer, last read before this iteration's barrier
    };
    for (int k = 0; k < nzc; k += 3) {
        plane(k, Ym, Yc, Yp, Pm, Pc, Pp);
        if (k + 1 < nzc) plane(k + 1, Yc, Yp, Ym, Pc, Pp, Pm);
        if (k + 2 < nzc) plane(k + 2, Yp, Ym, Yc, Pp, Pm, Pc);
    }
}

}  // namespace tcp
