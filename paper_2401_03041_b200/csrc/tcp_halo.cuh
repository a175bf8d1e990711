// Ghost-plane traffic of a z-slab (block decomposition of Algorithm 1): what a slab's
// neighbour needs from its boundary plane, gathered into one message per face and scattered on arrival.
//
// With the SoA layout [q][z][y][x] one z-plane of one population is contiguous, so a message is a list of
// plane copies: the 9 populations of h~ and of g~ that cross the face, the crossing populations of f~
// (1, 5, 5, 9 for D3Q7/15/19/27), and the phi and T planes the 27-point stencils of the neighbour's
// boundary cells read.  u is only ever read by its own cell and does not travel.
#pragma once
#include <cuda_runtime.h>

#include "tcp_lattice.cuh"

namespace tcp {

constexpr int kHaloMaxPlanes = 64;   // two faces x (9 + 9 + 9 + 2)

struct HaloCopy {
    const void* src[kHaloMaxPlanes];
    void* dst[kHaloMaxPlanes];
    int nplanes;
    int plane_cells;
};

template <typename real>
__global__ void __launch_bounds__(256) halo_copy_kernel(const HaloCopy C) {
    const int i = blockIdx.x * 256 + threadIdx.x;
    if (i >= C.plane_cells) return;
    const real* __restrict__ s = static_cast<const real*>(C.src[blockIdx.y]);
    real* __restrict__ d = static_cast<real*>(C.dst[blockIdx.y]);
    d[i] = s[i];
}

// number of populations of stencil Q (0 = none) whose c_z equals dir
inline int halo_crossing(int Q, int dir) {
    int n = 0;
    for (int k = 0; k < Q; ++k)
        if (cz27(q_of(Q, k)) == dir) ++n;
    return n;
}

}  // namespace tcp
