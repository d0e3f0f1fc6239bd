// packed_f32.cuh -- two fp32 lanes in one 64-bit register pair, for the sm_100 packed instructions FFMA2 / FADD2 / FMUL2
// (PTX fma.rn.f32x2 ..., CUDA's __ffma2_rn ...).
//
// A 3-register scalar FFMA issues every second cycle per SM sub-partition on Blackwell (B300_MICROARCH.md, "Pipe rates");
// the packed form does two FMAs per lane in the same slot, so a kernel bound by fp32 FMA issue -- the two-index and
// adjoint representations applied on the fly from the fundamental link, 230 FMA per half-spinor component and hop -- halves
// its FMA instruction count when the TWO half-spinor components of a hop ride in the two lanes: both are multiplied by
// the same link, which is broadcast once per hop.  Each lane rounds exactly like the scalar fmaf/+/*; the packed kernel
// differs from the scalar one only where the compiler contracts a scalar a*b+c that is written here as FMUL2 then FADD2.
//
// `pk::f32x2` models just enough of an arithmetic type for the link multiplies of dphi_kernel.cuh to be instantiated with
// Real = f32x2: broadcast from a scalar, + - * unary minus, *=, +=, and fma (found by argument-dependent lookup).
#pragma once
#include <cuda_runtime.h>

namespace hr {
namespace pk {

struct f32x2 {
    float2 v;
    f32x2() = default;
    __host__ __device__ constexpr f32x2(float s) : v{ s, s } {}            // broadcast
    __host__ __device__ constexpr f32x2(float lo, float hi) : v{ lo, hi } {}
    __host__ __device__ constexpr explicit f32x2(float2 p) : v{ p.x, p.y } {}
};

__device__ __forceinline__ f32x2 fma(f32x2 a, f32x2 b, f32x2 c) { return f32x2(__ffma2_rn(a.v, b.v, c.v)); }
__device__ __forceinline__ f32x2 operator*(f32x2 a, f32x2 b) { return f32x2(__fmul2_rn(a.v, b.v)); }
__device__ __forceinline__ f32x2 operator+(f32x2 a, f32x2 b) { return f32x2(__fadd2_rn(a.v, b.v)); }
// lane-wise negation / subtraction: sign flips are exact, so a - b == a + (-b) bit for bit
__device__ __forceinline__ f32x2 operator-(f32x2 a) { return f32x2(-a.v.x, -a.v.y); }
__device__ __forceinline__ f32x2 operator-(f32x2 a, f32x2 b) { return f32x2(__fadd2_rn(a.v, (-b).v)); }
__device__ __forceinline__ f32x2 &operator*=(f32x2 &a, f32x2 b) { a = a * b; return a; }
__device__ __forceinline__ f32x2 &operator+=(f32x2 &a, f32x2 b) { a = a + b; return a; }

} // namespace pk
} // namespace hr
