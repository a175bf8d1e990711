// fused step kernels, double, wall variants (see tcp_launch.inl)
#define TCP_REAL double
#define TCP_WALLS_ONLY 1
#include "tcp_launch.inl"
