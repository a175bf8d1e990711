// Arithmetic types of the kernels.
//
//   double, float   one cell per thread
//   f32x2           two x-adjacent cells per thread in packed single precision: sm_100 has FADD2 / FMUL2 /
//                   FFMA2 (two fp32 lanes per instruction; nvcc contracts __fmul2_rn + __fadd2_rn into
//                   FFMA2), so the collisions of a pair cost the instructions of one fp64 cell.  All
//                   collision code is written once, against `real`, and instantiated with any of the three.
//   wide_t<real>    what the zeroth moment is summed in by the single-precision variants
#pragma once
#include <cuda_runtime.h>

namespace tcp {

struct f32x2 {
    float2 v;
    f32x2() = default;
    __host__ __device__ __forceinline__ f32x2(float a, float b) : v{a, b} {}
    template <typename S, typename = decltype(static_cast<float>(S()))>
    __host__ __device__ __forceinline__ f32x2(S a) : v{static_cast<float>(a), static_cast<float>(a)} {}   // broadcast
};
__device__ __forceinline__ f32x2 operator+(f32x2 a, f32x2 b) { f32x2 r; r.v = __fadd2_rn(a.v, b.v); return r; }
__device__ __forceinline__ f32x2 operator*(f32x2 a, f32x2 b) { f32x2 r; r.v = __fmul2_rn(a.v, b.v); return r; }
__device__ __forceinline__ f32x2 operator-(f32x2 a) { return f32x2(-a.v.x, -a.v.y); }
__device__ __forceinline__ f32x2 operator-(f32x2 a, f32x2 b) { return a + (-b); }
__device__ __forceinline__ f32x2 operator/(f32x2 a, f32x2 b) { return f32x2(a.v.x / b.v.x, a.v.y / b.v.y); }
__device__ __forceinline__ f32x2& operator+=(f32x2& a, f32x2 b) { a = a + b; return a; }
__device__ __forceinline__ f32x2& operator-=(f32x2& a, f32x2 b) { a = a - b; return a; }
__device__ __forceinline__ f32x2& operator*=(f32x2& a, f32x2 b) { a = a * b; return a; }

struct f64x2 {
    double x, y;
};
__device__ __forceinline__ f64x2& operator+=(f64x2& a, f64x2 b) { a.x += b.x; a.y += b.y; return a; }
__device__ __forceinline__ f64x2& operator-=(f64x2& a, f64x2 b) { a.x -= b.x; a.y -= b.y; return a; }

template <typename real> struct real_traits;
template <> struct real_traits<double> { using scalar = double; using wide = double; static constexpr bool single = false; static constexpr int lanes = 1; };
template <> struct real_traits<float>  { using scalar = float;  using wide = double; static constexpr bool single = true;  static constexpr int lanes = 1; };
template <> struct real_traits<f32x2>  { using scalar = float;  using wide = f64x2;  static constexpr bool single = true;  static constexpr int lanes = 2; };
template <typename real> using wide_t = typename real_traits<real>::wide;
template <typename real> using scalar_t = typename real_traits<real>::scalar;

__device__ __forceinline__ double widen(double a) { return a; }
__device__ __forceinline__ double widen(float a) { return (double)a; }
__device__ __forceinline__ f64x2 widen(f32x2 a) { return f64x2{(double)a.v.x, (double)a.v.y}; }
template <typename real> __device__ __forceinline__ real narrow(wide_t<real> a);
template <> __device__ __forceinline__ double narrow<double>(double a) { return a; }
template <> __device__ __forceinline__ float narrow<float>(double a) { return (float)a; }
template <> __device__ __forceinline__ f32x2 narrow<f32x2>(f64x2 a) { return f32x2((float)a.x, (float)a.y); }
template <typename real> __device__ __forceinline__ wide_t<real> wide_zero() { return wide_t<real>{}; }

template <typename real> __device__ __forceinline__ real rsqrt_(real x);
template <> __device__ __forceinline__ double rsqrt_<double>(double x) { return 1.0 / sqrt(x); }
template <> __device__ __forceinline__ float rsqrt_<float>(float x) { return 1.0f / sqrtf(x); }
template <> __device__ __forceinline__ f32x2 rsqrt_<f32x2>(f32x2 x) { return f32x2(1.0f / sqrtf(x.v.x), 1.0f / sqrtf(x.v.y)); }

}  // namespace tcp
