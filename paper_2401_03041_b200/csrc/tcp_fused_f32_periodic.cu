// fused step kernels, float, periodic variants (see tcp_launch.inl)
#define TCP_REAL float
#define TCP_PAIR 1
#include "tcp_launch.inl"
