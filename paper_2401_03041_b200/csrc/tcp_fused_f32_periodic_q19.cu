// fused step kernels, float, periodic variants, D3Q19 hydrodynamic lattice (see tcp_launch.inl)
#define TCP_REAL float
#define TCP_QH 19
#define TCP_PAIR 1
#include "tcp_launch.inl"
