// fused_step_rows_kernel: the same fused step as fused_step_kernel, but a block owns one segment
// of one x-row and the 27 + 27 + Q_T population rows it pulls from are staged in shared memory by
// the TMA (cp.async.bulk, one bulk copy per row, completion on an mbarrier), so the bytes in flight
// per SM no longer depend on registers x resident warps.
//
// Geometry.  A row of direction q that the segment [x0, x0+len) of row (y,z) pulls from is the
// contiguous piece [x0 - c_x, x0 - c_x + len) of row (y - c_y, z - c_z) of plane q (periodic wrap in
// y, z; halfway bounce-back at a y / z wall replaces it by the segment's own piece of plane opp(q)).
// cp.async.bulk needs 16-byte aligned addresses and sizes, so every row is fetched as the aligned
// window [x0 - A, x0 + L + A), A = 16 B / sizeof(real) elements, and read at offset A - c_x; windows
// that stick out of the row get their wrapped ends by two 16-byte copies.  Requirements (checked
// on the host, otherwise the flat kernel runs): x periodic, nx a multiple of A.
#pragma once
#include <cstdint>

#include "tcp_step.cuh"

namespace tcp {

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void fence_mbar_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    uint32_t done;
    do {
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(done)
                     : "r"(smem_u32(bar)), "r"(parity)
                     : "memory");
    } while (!done);
}

template <typename real>
struct RowGeom {
    static constexpr int A = 16 / (int)sizeof(real);   // halo elements on each side of the window
};

// Issue the bulk copies of one row window.  dst: shared row (P = L + 2A elements), plane: global
// plane of the direction to read, rowbase: element offset of the source row's x = 0.
template <typename real>
__device__ __forceinline__ void stage_row(real* dst, const real* plane, long long rowbase, int x0, int len, int nx, uint64_t* bar) {
    constexpr int A = RowGeom<real>::A;
    const int es = (int)sizeof(real);
    const int lo = x0 - A, hi = x0 + len + A;            // needed source range [lo, hi)
    const int mlo = lo < 0 ? 0 : lo, mhi = hi > nx ? nx : hi;
    bulk_g2s(dst + (mlo - lo), plane + rowbase + mlo, (uint32_t)((mhi - mlo) * es), bar);
    if (lo < 0) bulk_g2s(dst, plane + rowbase + (nx - A), 16u, bar);                 // x = -A .. -1 wraps to the row's end
    if (hi > nx) bulk_g2s(dst + (nx - lo), plane + rowbase, 16u, bar);               // x = nx .. nx+A-1 wraps to its start
}
__device__ __forceinline__ uint32_t row_bytes(int len, int A, int es) { return (uint32_t)((len + 2 * A) * es); }

// block-level source row of direction (cy, cz) for the segment's row (y, z): wrapped row offset, or
// bounce = true when the link crosses a y / z wall
__device__ __forceinline__ long long source_row(int y, int z, int cy, int cz, int nx, int ny, int nz, bool wy, bool wz, bool& bounce) {
    int ys = y - cy, zs = z - cz;
    bounce = false;
    if (ys < 0) { if (wy) bounce = true; else ys += ny; }
    else if (ys >= ny) { if (wy) bounce = true; else ys -= ny; }
    if (zs < 0) { if (wz) bounce = true; else zs += nz; }
    else if (zs >= nz) { if (wz) bounce = true; else zs -= nz; }
    if (bounce) { ys = y; zs = z; }
    return (long long)nx * (ys + (long long)ny * zs);
}

// blockDim.x = Lseg rounded up to a warp, at most TCP_ROWS_MAXT
#ifndef TCP_ROWS_MAXT
#define TCP_ROWS_MAXT 128
#endif
#ifndef TCP_ROWS_MINB
#define TCP_ROWS_MINB 3
#endif
constexpr int kRowsMaxThreads = TCP_ROWS_MAXT;

template <typename real, int QT, bool WALLS>
__global__ void __launch_bounds__(TCP_ROWS_MAXT, TCP_ROWS_MINB) fused_step_rows_kernel(const StepArgs<real> A_, int Lseg) {
    constexpr int MODE = 0;
    constexpr int AH = RowGeom<real>::A;
    const StepArgs<real>& A = A_;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int P = Lseg + 2 * AH;
    real* rows = reinterpret_cast<real*>(smem_raw);                       // [27 + 27 + QT][P]
    uint64_t* bars = reinterpret_cast<uint64_t*>(rows + (size_t)(54 + QT) * P);   // 3 mbarriers

    const int tid = threadIdx.x;
    const int x0 = blockIdx.x * Lseg;
    const int y = blockIdx.y, z = blockIdx.z;
    const int len = min(Lseg, A.nx - x0);
    const long long N = A.ncell;
    const bool wy = WALLS && A.wall[1], wz = WALLS && A.wall[2];

    if (tid == 0) {
        mbar_init(&bars[0], 1); mbar_init(&bars[1], 1); mbar_init(&bars[2], 1);
        fence_mbar_init();
    }
    __syncthreads();
    if (tid == 0) {
        const uint32_t rb = row_bytes(len, AH, (int)sizeof(real));
        mbar_arrive_expect_tx(&bars[0], 27u * rb);
#pragma unroll 1
        for (int q = 0; q < 27; ++q) {
            bool bounce;
            const long long rowbase = source_row(y, z, cy27(q), cz27(q), A.nx, A.ny, A.nz, wy, wz, bounce);
            stage_row<real>(rows + (size_t)q * P, A.h_in + (bounce ? 26 - q : q) * N, rowbase, x0, len, A.nx, &bars[0]);
        }
        mbar_arrive_expect_tx(&bars[1], 27u * rb);
#pragma unroll 1
        for (int q = 0; q < 27; ++q) {
            bool bounce;
            const long long rowbase = source_row(y, z, cy27(q), cz27(q), A.nx, A.ny, A.nz, wy, wz, bounce);
            stage_row<real>(rows + (size_t)(27 + q) * P, A.g_in + (bounce ? 26 - q : q) * N, rowbase, x0, len, A.nx, &bars[1]);
        }
        if constexpr (QT > 0) {
            mbar_arrive_expect_tx(&bars[2], (uint32_t)QT * rb);
            static_for<0, QT>([&](auto K) {
                constexpr int k = decltype(K)::value, q = q_of(QT, k);
                bool bounce;
                const long long rowbase = source_row(y, z, cy27(q), cz27(q), A.nx, A.ny, A.nz, wy, wz, bounce);
                stage_row<real>(rows + (size_t)(54 + k) * P, A.f_in + (bounce ? QT - 1 - k : k) * N, rowbase, x0, len, A.nx, &bars[2]);
            });
        }
    }

    const bool active = tid < len;
    const int t = active ? tid : 0;          // lanes past the segment's end shadow lane 0 and store nothing
    const int x = x0 + t;
    Nbh<WALLS> nb;
    nb.init_xyz(A, x, y, z);
    const int cell = nb.idx;

    real phi_c, G[3], lapPhi, T_c, Th[3], lapT;
    stencil27<real, WALLS, false>(A, nb, A.phi_in, phi_c, G, lapPhi);
    stencil27<real, WALLS, true>(A, nb, A.T_in, T_c, Th, lapT);
    real u[3] = {A.u[cell], A.u[N + cell], A.u[2 * N + cell]};

    // pulled value of direction q from its staged row: shifted by -c_x, or unshifted on a bounce row
    auto staged = [&](int row, int q27i) -> real {
        const int cx = cx27(q27i), cy = cy27(q27i), cz = cz27(q27i);
        bool bounce = false;
        if (WALLS) bounce = (cy == 1 && nb.lo[1]) || (cy == -1 && nb.hi[1]) || (cz == 1 && nb.lo[2]) || (cz == -1 && nb.hi[2]);
        return rows[(size_t)row * P + t + AH - (bounce ? 0 : cx)];
    };

    real phi_new;
    {
        mbar_wait(&bars[0], 0);
        real h[27];
#pragma unroll
        for (int q = 0; q < 27; ++q) h[q] = staged(q, q);
        phi_new = collide_phase<real, MODE>(A, h, G, phi_c, u);
        if (active) {
#pragma unroll
            for (int q = 0; q < 27; ++q) A.h_out[q * N + cell] = h[q];
            A.phi_out[cell] = phi_new;
        }
    }
    {
        mbar_wait(&bars[1], 0);
        real g[27];
#pragma unroll
        for (int q = 0; q < 27; ++q) g[q] = staged(27 + q, q);
        collide_hydro<real, MODE>(A, g, phi_c, G, lapPhi, T_c, Th, u);
        if (active) {
#pragma unroll
            for (int q = 0; q < 27; ++q) A.g_out[q * N + cell] = g[q];
            A.u[cell] = u[0]; A.u[N + cell] = u[1]; A.u[2 * N + cell] = u[2];
        }
    }
    if constexpr (QT > 0) {
        mbar_wait(&bars[2], 0);
        real f[QT];
        static_for<0, QT>([&](auto K) {
            constexpr int k = decltype(K)::value, q = q_of(QT, k);
            constexpr int cx = cx27(q), cy = cy27(q), cz = cz27(q);
            int face = 0;
            const int ax = nb.crossed(-cx, -cy, -cz, face);
            if (WALLS && ax >= 0)   // anti-bounce-back: the staged row is plane opp(k), own row, unshifted
                f[k] = real(2.0 * weight(QT, cls27(q))) * wall_temperature(A, nb, ax, face, -cx, -cy, -cz) - rows[(size_t)(54 + k) * P + t + AH];
            else
                f[k] = rows[(size_t)(54 + k) * P + t + AH - cx];
        });
        const real qT = A.q_src ? A.q_src[cell] : real(0);
        const real Tn = collide_thermal<real, QT, MODE>(A, f, phi_new, u, qT);
        if (active) {
            static_for<0, QT>([&](auto K) { constexpr int k = decltype(K)::value; A.f_out[k * N + cell] = f[k]; });
            A.T_out[cell] = Tn;
        }
    }
}

}  // namespace tcp
