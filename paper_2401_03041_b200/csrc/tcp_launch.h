// Launchers of the fused step kernels, one translation unit per precision so that the ~70 template
// instantiations compile in parallel (paper_2401_03041_b200/build.py).
#pragma once
#include <cuda_runtime.h>

#include "tcp_device.cuh"

namespace tcp {

constexpr int kMaxDevices = 64;

struct FusedCfg {
    int qt;          // thermal stencil size, 0 on the Runge-Kutta paths
    bool walls;      // any WALLS axis
    int mode;        // 0 closed-form central moments, 1 BGK, 2 general rates, 3 calibration, 4 = 0 with the Maxwellian equilibrium
    int aa;          // 0 two-grid; AA in-place streaming: 1 even step, 2 odd step
    int device;      // CUDA device of the simulation (per-device kernel attributes)
    unsigned grid;
};

cudaError_t launch_fused_periodic(const FusedCfg& c, const StepArgs<double>& A, cudaStream_t stream);
cudaError_t launch_fused_periodic(const FusedCfg& c, const StepArgs<float>& A, cudaStream_t stream);
cudaError_t launch_fused_walls(const FusedCfg& c, const StepArgs<double>& A, cudaStream_t stream);
cudaError_t launch_fused_walls(const FusedCfg& c, const StepArgs<float>& A, cudaStream_t stream);

// single precision, two cells per thread, packed arithmetic (tcp_pair.cuh): x periodic and nx even only
cudaError_t launch_pair_periodic(const FusedCfg& c, const StepArgs<float>& A, cudaStream_t stream);
cudaError_t launch_pair_walls(const FusedCfg& c, const StepArgs<float>& A, cudaStream_t stream);

// the same with the D3Q19 hydrodynamic lattice (tcp_params::hydro_lattice = 19; c.mode 0 or 1 only)
cudaError_t launch_fused_periodic_q19(const FusedCfg& c, const StepArgs<double>& A, cudaStream_t stream);
cudaError_t launch_fused_periodic_q19(const FusedCfg& c, const StepArgs<float>& A, cudaStream_t stream);
cudaError_t launch_fused_walls_q19(const FusedCfg& c, const StepArgs<double>& A, cudaStream_t stream);
cudaError_t launch_fused_walls_q19(const FusedCfg& c, const StepArgs<float>& A, cudaStream_t stream);
cudaError_t launch_pair_periodic_q19(const FusedCfg& c, const StepArgs<float>& A, cudaStream_t stream);
cudaError_t launch_pair_walls_q19(const FusedCfg& c, const StepArgs<float>& A, cudaStream_t stream);

// thermal LB update alone (tcp_relax_temperature); c.mode 0 / 1, c.aa as above
cudaError_t launch_thermal_periodic(const FusedCfg& c, const StepArgs<double>& A, cudaStream_t stream);
cudaError_t launch_thermal_periodic(const FusedCfg& c, const StepArgs<float>& A, cudaStream_t stream);
cudaError_t launch_thermal_walls(const FusedCfg& c, const StepArgs<double>& A, cudaStream_t stream);
cudaError_t launch_thermal_walls(const FusedCfg& c, const StepArgs<float>& A, cudaStream_t stream);

}  // namespace tcp
