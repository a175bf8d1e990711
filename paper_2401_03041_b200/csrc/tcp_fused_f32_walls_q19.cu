// fused step kernels, float, walls variants, D3Q19 hydrodynamic lattice (see tcp_launch.inl)
#define TCP_REAL float
#define TCP_QH 19
#define TCP_PAIR 1
#define TCP_WALLS_ONLY 1
#include "tcp_launch.inl"
