// Included by the tcp_fused_*.cu translation units with TCP_REAL defined (and TCP_WALLS_ONLY, TCP_PAIR, TCP_QH).
// TCP_QH = 19 builds the kernels of the D3Q19 hydrodynamic lattice under the names launch_*_q19 (closed-form central-moment
// and BGK collisions only; no calibration kernel, no thermal-only kernel: those do not depend on the hydrodynamic lattice).
#ifndef TCP_QH
#define TCP_QH 27
#endif
#include "tcp_launch.h"
#include "tcp_step.cuh"
#ifdef TCP_PAIR
#include "tcp_pair.cuh"
#endif

namespace tcp {
namespace {

template <typename real, int QT, bool WALLS, int MODE, int AA>
cudaError_t launch_staged(const FusedCfg& c, const StepArgs<real>& A, cudaStream_t stream) {
    const size_t smem = (size_t)(27 + TCP_QH + QT - (h_direct<real, QT, AA>() ? 27 : 0)) * kBlock * sizeof(real);
    auto kern = fused_step_async_kernel<real, QT, WALLS, MODE, AA, TCP_QH>;
    static bool configured[kMaxDevices] = {};   // once per instantiation and device: saves ~1 us per launch
    if (!configured[c.device]) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        configured[c.device] = true;
    }
    kern<<<c.grid, kBlock, smem, stream>>>(A);
    return cudaGetLastError();
}

template <typename real, int QT, bool WALLS>
cudaError_t dispatch(const FusedCfg& c, const StepArgs<real>& A, cudaStream_t stream) {
#if TCP_QH == 27
    if (c.mode == 3) {   // roofline calibration kernel (tcp_pattern_copy_ms): two-grid, periodic only
        if constexpr (!WALLS) return launch_staged<real, QT, false, 3, 0>(c, A, stream);
        else return cudaErrorNotSupported;
    }
#endif
#if TCP_QH == 27
    if (c.mode == 4) {   // Maxwellian equilibrium: D3Q27 lattices only (thermal D3Q27 LB or a Runge-Kutta path)
        if constexpr (QT == 0 || QT == 27) {
            switch (c.aa) {
            case 0: return launch_staged<real, QT, WALLS, 4, 0>(c, A, stream);
            case 1: return launch_staged<real, QT, WALLS, 4, 1>(c, A, stream);
            default: return launch_staged<real, QT, WALLS, 4, 2>(c, A, stream);
            }
        } else return cudaErrorNotSupported;
    }
#endif
    switch (3 * c.aa + c.mode) {   // c.aa: 0 two-grid, 1 AA even step, 2 AA odd step
    case 0: return launch_staged<real, QT, WALLS, 0, 0>(c, A, stream);
    case 1: return launch_staged<real, QT, WALLS, 1, 0>(c, A, stream);
    case 3: return launch_staged<real, QT, WALLS, 0, 1>(c, A, stream);
    case 4: return launch_staged<real, QT, WALLS, 1, 1>(c, A, stream);
    case 6: return launch_staged<real, QT, WALLS, 0, 2>(c, A, stream);
    case 7: return launch_staged<real, QT, WALLS, 1, 2>(c, A, stream);
#if TCP_QH == 27   // general central-moment rates: tensor-product D3Q27 basis only
    case 2: return launch_staged<real, QT, WALLS, 2, 0>(c, A, stream);
    case 5: return launch_staged<real, QT, WALLS, 2, 1>(c, A, stream);
    case 8: return launch_staged<real, QT, WALLS, 2, 2>(c, A, stream);
#endif
    default: return cudaErrorNotSupported;
    }
}

template <typename real, bool WALLS>
cudaError_t by_stencil(const FusedCfg& c, const StepArgs<real>& A, cudaStream_t stream) {
    switch (c.qt) {
    case 7: return dispatch<real, 7, WALLS>(c, A, stream);
    case 15: return dispatch<real, 15, WALLS>(c, A, stream);
    case 19: return dispatch<real, 19, WALLS>(c, A, stream);
    case 27: return dispatch<real, 27, WALLS>(c, A, stream);
    default: return dispatch<real, 0, WALLS>(c, A, stream);
    }
}

#if TCP_QH == 27
template <typename real, int QT, bool WALLS>
cudaError_t thermal_dispatch(const FusedCfg& c, const StepArgs<real>& A, cudaStream_t stream) {
    if (c.mode == 4) {   // Maxwellian equilibrium (D3Q27 thermal LB only)
        if constexpr (QT == 27) {
            switch (c.aa) {
            case 0: thermal_only_kernel<real, QT, WALLS, 4, 0><<<c.grid, kBlock, 0, stream>>>(A); break;
            case 1: thermal_only_kernel<real, QT, WALLS, 4, 1><<<c.grid, kBlock, 0, stream>>>(A); break;
            default: thermal_only_kernel<real, QT, WALLS, 4, 2><<<c.grid, kBlock, 0, stream>>>(A); break;
            }
            return cudaGetLastError();
        } else return cudaErrorNotSupported;
    }
    switch (2 * c.aa + (c.mode == 1)) {
    case 0: thermal_only_kernel<real, QT, WALLS, 0, 0><<<c.grid, kBlock, 0, stream>>>(A); break;
    case 1: thermal_only_kernel<real, QT, WALLS, 1, 0><<<c.grid, kBlock, 0, stream>>>(A); break;
    case 2: thermal_only_kernel<real, QT, WALLS, 0, 1><<<c.grid, kBlock, 0, stream>>>(A); break;
    case 3: thermal_only_kernel<real, QT, WALLS, 1, 1><<<c.grid, kBlock, 0, stream>>>(A); break;
    case 4: thermal_only_kernel<real, QT, WALLS, 0, 2><<<c.grid, kBlock, 0, stream>>>(A); break;
    default: thermal_only_kernel<real, QT, WALLS, 1, 2><<<c.grid, kBlock, 0, stream>>>(A); break;
    }
    return cudaGetLastError();
}
template <typename real, bool WALLS>
cudaError_t thermal_by_stencil(const FusedCfg& c, const StepArgs<real>& A, cudaStream_t stream) {
    switch (c.qt) {
    case 7: return thermal_dispatch<real, 7, WALLS>(c, A, stream);
    case 15: return thermal_dispatch<real, 15, WALLS>(c, A, stream);
    case 19: return thermal_dispatch<real, 19, WALLS>(c, A, stream);
    case 27: return thermal_dispatch<real, 27, WALLS>(c, A, stream);
    default: return cudaErrorInvalidValue;
    }
}
#endif

#ifdef TCP_PAIR
// packed-pair single-precision kernels (tcp_pair.cuh)
template <int QT, bool WALLS, int MODE, int AA>
cudaError_t launch_pair(const FusedCfg& c, const StepArgs<f32x2>& A, cudaStream_t stream) {
    const size_t smem = (size_t)(27 + TCP_QH + QT - (pair_h_direct<QT, AA>() ? 27 : 0)) * kBlock * sizeof(float2);
    auto kern = fused_step_pair_kernel<QT, WALLS, MODE, AA, TCP_QH>;
    static bool configured[kMaxDevices] = {};
    if (!configured[c.device]) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        configured[c.device] = true;
    }
    const unsigned grid = (unsigned)((((A.cell1 - A.cell0) >> 1) + kBlock - 1) / kBlock);
    kern<<<grid, kBlock, smem, stream>>>(A);
    return cudaGetLastError();
}
template <int QT, bool WALLS>
cudaError_t pair_dispatch(const FusedCfg& c, const StepArgs<f32x2>& A, cudaStream_t stream) {
#if TCP_QH == 27
    if (c.mode == 4) {
        if constexpr (QT == 0 || QT == 27) {
            switch (c.aa) {
            case 0: return launch_pair<QT, WALLS, 4, 0>(c, A, stream);
            case 1: return launch_pair<QT, WALLS, 4, 1>(c, A, stream);
            default: return launch_pair<QT, WALLS, 4, 2>(c, A, stream);
            }
        } else return cudaErrorNotSupported;
    }
#endif
    switch (c.aa) {   // closed-form collision modes only (BGK and general rates run the scalar kernels)
    case 0: return launch_pair<QT, WALLS, 0, 0>(c, A, stream);
    case 1: return launch_pair<QT, WALLS, 0, 1>(c, A, stream);
    default: return launch_pair<QT, WALLS, 0, 2>(c, A, stream);
    }
}
template <bool WALLS>
cudaError_t pair_by_stencil(const FusedCfg& c, const StepArgs<float>& Af, cudaStream_t stream) {
    const StepArgs<f32x2> A(Af);
    switch (c.qt) {
    case 7: return pair_dispatch<7, WALLS>(c, A, stream);
    case 15: return pair_dispatch<15, WALLS>(c, A, stream);
    case 19: return pair_dispatch<19, WALLS>(c, A, stream);
    case 27: return pair_dispatch<27, WALLS>(c, A, stream);
    default: return pair_dispatch<0, WALLS>(c, A, stream);
    }
}
#endif

}  // namespace

#if TCP_QH == 27
#define TCP_NAME(n) n
#else
#define TCP_NAME(n) n##_q19
#endif

#ifdef TCP_PAIR
#ifdef TCP_WALLS_ONLY
cudaError_t TCP_NAME(launch_pair_walls)(const FusedCfg& c, const StepArgs<float>& A, cudaStream_t stream) { return pair_by_stencil<true>(c, A, stream); }
#else
cudaError_t TCP_NAME(launch_pair_periodic)(const FusedCfg& c, const StepArgs<float>& A, cudaStream_t stream) { return pair_by_stencil<false>(c, A, stream); }
#endif
#endif

#ifdef TCP_WALLS_ONLY
cudaError_t TCP_NAME(launch_fused_walls)(const FusedCfg& c, const StepArgs<TCP_REAL>& A, cudaStream_t stream) { return by_stencil<TCP_REAL, true>(c, A, stream); }
#if TCP_QH == 27
cudaError_t launch_thermal_walls(const FusedCfg& c, const StepArgs<TCP_REAL>& A, cudaStream_t stream) { return thermal_by_stencil<TCP_REAL, true>(c, A, stream); }
#endif
#else
cudaError_t TCP_NAME(launch_fused_periodic)(const FusedCfg& c, const StepArgs<TCP_REAL>& A, cudaStream_t stream) { return by_stencil<TCP_REAL, false>(c, A, stream); }
#if TCP_QH == 27
cudaError_t launch_thermal_periodic(const FusedCfg& c, const StepArgs<TCP_REAL>& A, cudaStream_t stream) { return thermal_by_stencil<TCP_REAL, false>(c, A, stream); }
#endif
#endif

}  // namespace tcp
