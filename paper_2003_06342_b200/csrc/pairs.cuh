// Two x-adjacent nodes per thread in single precision: the value types node_update is instantiated with when a thread
// carries a PAIR of nodes.  f2 is two floats in one 64-bit register pair; its arithmetic is the packed single-precision
// instructions of sm_100 (add / mul / fma .f32x2 -> FADD2 / FMUL2 / FFMA2: one issue slot for both nodes).  A product is kept lazy
// (f2prod) until it meets a sum, so that a * b + c becomes ONE packed fma, as the compiler contracts it for scalars.
// d2 is two doubles (the phase-field path stays wide); plain member-wise arithmetic, which the compiler
// contracts itself.
#pragma once

#include <cuda_runtime.h>

namespace lbm {

struct f2 {
    float x, y;
    f2() = default;
    __host__ __device__ constexpr f2(float a, float b) : x(a), y(b) {}
    __host__ __device__ constexpr explicit f2(float a) : x(a), y(a) {}
    __host__ __device__ constexpr explicit f2(double a) : x((float)a), y((float)a) {}
    __host__ __device__ constexpr explicit f2(int a) : x((float)a), y((float)a) {}
    __host__ __device__ constexpr f2 operator-() const { return f2(-x, -y); }
};

#ifdef __CUDACC__
__device__ __forceinline__ float2 as_float2(f2 a) { return make_float2(a.x, a.y); }
__device__ __forceinline__ f2 as_f2(float2 a) { return f2(a.x, a.y); }
__device__ __forceinline__ f2 add2(f2 a, f2 b) { return as_f2(__fadd2_rn(as_float2(a), as_float2(b))); }
__device__ __forceinline__ f2 mul2(f2 a, f2 b) { return as_f2(__fmul2_rn(as_float2(a), as_float2(b))); }
__device__ __forceinline__ f2 fma2(f2 a, f2 b, f2 c) { return as_f2(__ffma2_rn(as_float2(a), as_float2(b), as_float2(c))); }

struct f2prod {   // a * b, not yet evaluated
    f2 a, b;
    __device__ __forceinline__ operator f2() const { return mul2(a, b); }
    __device__ __forceinline__ f2prod operator-() const { return f2prod{-a, b}; }
};

__device__ __forceinline__ f2prod operator*(f2 a, f2 b) { return f2prod{a, b}; }
__device__ __forceinline__ f2prod operator*(f2prod p, f2 c) { return f2prod{mul2(p.a, p.b), c}; }
__device__ __forceinline__ f2prod operator*(f2 c, f2prod p) { return f2prod{c, mul2(p.a, p.b)}; }
__device__ __forceinline__ f2prod operator*(f2prod p, f2prod q) { return f2prod{mul2(p.a, p.b), mul2(q.a, q.b)}; }
__device__ __forceinline__ f2 operator+(f2 a, f2 b) { return add2(a, b); }
__device__ __forceinline__ f2 operator-(f2 a, f2 b) { return add2(a, -b); }
__device__ __forceinline__ f2 operator+(f2prod p, f2 c) { return fma2(p.a, p.b, c); }
__device__ __forceinline__ f2 operator+(f2 c, f2prod p) { return fma2(p.a, p.b, c); }
__device__ __forceinline__ f2 operator-(f2prod p, f2 c) { return fma2(p.a, p.b, -c); }
__device__ __forceinline__ f2 operator-(f2 c, f2prod p) { return fma2(-p.a, p.b, c); }
__device__ __forceinline__ f2 operator+(f2prod p, f2prod q) { return fma2(p.a, p.b, mul2(q.a, q.b)); }
__device__ __forceinline__ f2 operator-(f2prod p, f2prod q) { return fma2(-q.a, q.b, mul2(p.a, p.b)); }
__device__ __forceinline__ f2 &operator+=(f2 &a, f2 b) { a = add2(a, b); return a; }
__device__ __forceinline__ f2 &operator-=(f2 &a, f2 b) { a = add2(a, -b); return a; }
__device__ __forceinline__ f2 &operator+=(f2 &a, f2prod p) { a = fma2(p.a, p.b, a); return a; }
__device__ __forceinline__ f2 &operator-=(f2 &a, f2prod p) { a = fma2(-p.a, p.b, a); return a; }
__device__ __forceinline__ f2 &operator*=(f2 &a, f2 b) { a = mul2(a, b); return a; }
__device__ __forceinline__ f2 operator/(f2 a, f2 b) { return f2(a.x / b.x, a.y / b.y); }

struct d2 {
    double x, y;
    d2() = default;
    __device__ constexpr d2(double a, double b) : x(a), y(b) {}
    __device__ constexpr explicit d2(double a) : x(a), y(a) {}
    __device__ constexpr explicit d2(f2 a) : x((double)a.x), y((double)a.y) {}
    __device__ constexpr d2 operator-() const { return d2(-x, -y); }
    __device__ explicit operator f2() const { return f2((float)x, (float)y); }
};
__device__ __forceinline__ d2 operator+(d2 a, d2 b) { return d2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ d2 operator-(d2 a, d2 b) { return d2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ d2 operator*(d2 a, d2 b) { return d2(a.x * b.x, a.y * b.y); }
#endif

}  // namespace lbm
