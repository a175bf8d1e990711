// fused step kernels, double, periodic variants, D3Q19 hydrodynamic lattice (see tcp_launch.inl)
#define TCP_REAL double
#define TCP_QH 19
#include "tcp_launch.inl"
