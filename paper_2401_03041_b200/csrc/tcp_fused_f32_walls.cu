// fused step kernels, float, wall variants (see tcp_launch.inl)
#define TCP_REAL float
#define TCP_PAIR 1
#define TCP_WALLS_ONLY 1
#include "tcp_launch.inl"
