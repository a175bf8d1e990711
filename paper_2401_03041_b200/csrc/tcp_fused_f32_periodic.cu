// fused step kernels, float, periodic variants (see tcp_launch.inl)
#define TCP_REAL float
#include "tcp_launch.inl"
