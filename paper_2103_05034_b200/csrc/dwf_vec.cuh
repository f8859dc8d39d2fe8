// dwf_vec.cuh -- lane-vector arithmetic for the native field layout.
//
// A "group" is the 16-byte unit of the native layout: one complex colour-spin component of VL
// adjacent fifth-dimension lanes:
//   fp32: VL = 2, group = float4  {re(s=2k), re(s=2k+1), im(s=2k), im(s=2k+1)}
//   fp64: VL = 1, group = double2 {re, im}
// All arithmetic on a group is done on V = float2 (two lanes, packed FFMA2/FADD2/FMUL2 of sm_100a,
// with the link element as the scalar-broadcast operand) or V = double.
#pragma once
#include <cuda_runtime.h>

namespace dwf {

template <typename R> struct Prec;
template <> struct Prec<float>  { using V = float2; using G = float4;  static constexpr int VL = 2; };
template <> struct Prec<double> { using V = double; using G = double2; static constexpr int VL = 1; };

// ---- packed fp32 (two lanes) ----
__device__ __forceinline__ float2 vzero(float2) { return make_float2(0.f, 0.f); }
__device__ __forceinline__ float2 vneg(float2 a) { return make_float2(-a.x, -a.y); }
__device__ __forceinline__ float2 vadd(float2 a, float2 b) { return __fadd2_rn(a, b); }
__device__ __forceinline__ float2 vsub(float2 a, float2 b) { return __fadd2_rn(a, make_float2(-b.x, -b.y)); }
__device__ __forceinline__ float2 vmul(float s, float2 b) { return __fmul2_rn(make_float2(s, s), b); }
__device__ __forceinline__ float2 vfma(float s, float2 b, float2 c) { return __ffma2_rn(make_float2(s, s), b, c); }
__device__ __forceinline__ float2 vfnma(float s, float2 b, float2 c) { return __ffma2_rn(make_float2(-s, -s), b, c); }
// lane-wise coefficient pair
__device__ __forceinline__ float2 vfma2(float2 s, float2 b, float2 c) { return __ffma2_rn(s, b, c); }
__device__ __forceinline__ float2 vswap(float2 a) { return make_float2(a.y, a.x); }
// s * (lanes swapped): two scalar multiplies that write the swapped positions (no register moves)
__device__ __forceinline__ float2 vswapmul(float s, float2 a) { return make_float2(s * a.y, s * a.x); }

// ---- fp64 (one lane) ----
__device__ __forceinline__ double vzero(double) { return 0.0; }
__device__ __forceinline__ double vneg(double a) { return -a; }
__device__ __forceinline__ double vadd(double a, double b) { return a + b; }
__device__ __forceinline__ double vsub(double a, double b) { return a - b; }
__device__ __forceinline__ double vmul(double s, double b) { return s * b; }
__device__ __forceinline__ double vfma(double s, double b, double c) { return fma(s, b, c); }
__device__ __forceinline__ double vfnma(double s, double b, double c) { return fma(-s, b, c); }
__device__ __forceinline__ double vfma2(double s, double b, double c) { return fma(s, b, c); }
__device__ __forceinline__ double vswap(double a) { return a; }
__device__ __forceinline__ double vswapmul(double s, double a) { return s * a; }

// complex number whose re and im are lane vectors
template <typename V> struct CV { V re, im; };

template <typename V> __device__ __forceinline__ CV<V> cadd(CV<V> a, CV<V> b) { return { vadd(a.re, b.re), vadd(a.im, b.im) }; }
template <typename V> __device__ __forceinline__ CV<V> csub(CV<V> a, CV<V> b) { return { vsub(a.re, b.re), vsub(a.im, b.im) }; }
// a + i b, a - i b
template <typename V> __device__ __forceinline__ CV<V> caddi(CV<V> a, CV<V> b) { return { vsub(a.re, b.im), vadd(a.im, b.re) }; }
template <typename V> __device__ __forceinline__ CV<V> csubi(CV<V> a, CV<V> b) { return { vadd(a.re, b.im), vsub(a.im, b.re) }; }

// ---- 16-byte group load / store ----
__device__ __forceinline__ CV<float2> unpack(float4 g) { return { make_float2(g.x, g.y), make_float2(g.z, g.w) }; }
__device__ __forceinline__ CV<double> unpack(double2 g) { return { g.x, g.y }; }
__device__ __forceinline__ float4 pack(CV<float2> c) { return make_float4(c.re.x, c.re.y, c.im.x, c.im.y); }
__device__ __forceinline__ double2 pack(CV<double> c) { return make_double2(c.re, c.im); }

// read-only (non-coherent) 128-bit load; data is never written by the same kernel
__device__ __forceinline__ float4 ldg_nc(const float4* p) { return __ldg(p); }
__device__ __forceinline__ double2 ldg_nc(const double2* p) { return __ldg(p); }
// plain load (buffer may alias the output of this kernel at the same address: read-then-write)
__device__ __forceinline__ float4 ld_plain(const float4* p) { return *p; }
__device__ __forceinline__ double2 ld_plain(const double2* p) { return *p; }

// Block index of (site, rhs) in a half field: sites come in groups of 2^sg_shift
// (one tile of the native site order); a group's blocks are ordered [rhs][site in group], so that the
// tile of one right-hand side is one contiguous run (a single bulk copy).
__device__ __forceinline__ long long blk_index(long long site, int r, int nrhs, int sg_shift) {
    const long long grp = site >> sg_shift;
    return ((grp * nrhs + r) << sg_shift) + (site - (grp << sg_shift));
}

}  // namespace dwf
