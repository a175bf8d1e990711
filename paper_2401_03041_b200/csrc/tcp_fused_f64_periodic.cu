// fused step kernels, double, periodic variants (see tcp_launch.inl)
#define TCP_REAL double
#include "tcp_launch.inl"
