// fused step kernels, double, walls variants, D3Q19 hydrodynamic lattice (see tcp_launch.inl)
#define TCP_REAL double
#define TCP_QH 19
#define TCP_WALLS_ONLY 1
#include "tcp_launch.inl"
