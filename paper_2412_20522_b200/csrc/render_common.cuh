// render_common.cuh -- pieces shared by the forward and backward blend kernels.
//
// Geometry of a block: one 16x16 tile, 64 threads = 2 warps.  A warp owns a 16x8
// pixel strip; a lane owns a 2x2 pixel quad, so the per-entry record read from shared memory and the
// row/column partial products are shared by 4 pixels, and (backward) 4 pixels are summed in
// registers before any cross-lane reduction.
//
// Per-entry record staged in shared memory (3 x float4).  The conic is pre-scaled into the log2
// domain and the opacity folded in as an offset, so that
//     log2(alpha) = e = lo + A2 dx^2 + B2 dx dy + C2 dy^2,   d = mean2d - pixel,
// and the alpha filter of the method (power > 0 or alpha < 1/255 => skip) becomes two compares on e
// BEFORE any exponential is taken:  e > lo  or  e < log2(1/255).
#pragma once
#include "mg_common.cuh"

#define RN_THREADS 64
#define RN_BATCH 128
#define RN_LOG2E 1.4426950408889634f
#define RN_LN2 0.6931471805599453f
#define RN_LOG2_ALPHA_MIN -7.994353436858858f  // log2(1/255)
#define RN_CULL_SLACK 1e-3f                    // warp-level cull keeps entries within 2^-10 of the threshold

struct RnRecord {
  float4 a;  // mx, my, A2, B2
  float4 b;  // C2, lo, mask, 1/o (backward) or unused
  float4 c;  // r, g, b, unused
};

__device__ __forceinline__ float rn_ex2(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ float rn_lg2(float x) {
  float y;
  asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}

struct RnRaw {  // attributes of one list entry as gathered from global memory
  float2 m2;
  float4 co;
  float r, g, b, m;
};

__device__ __forceinline__ RnRaw rn_gather(uint32_t id, const float2* __restrict__ means2d,
                                           const float4* __restrict__ conic_opacity, const float* __restrict__ rgb,
                                           const float* __restrict__ masks) {
  RnRaw v;
  v.m2 = __ldg(means2d + id);
  v.co = __ldg(conic_opacity + id);
  v.r = __ldg(rgb + 3 * (size_t)id);
  v.g = __ldg(rgb + 3 * (size_t)id + 1);
  v.b = __ldg(rgb + 3 * (size_t)id + 2);
  v.m = __ldg(masks + id);
  return v;
}

__device__ __forceinline__ RnRecord rn_make_record(const RnRaw& v) {
  RnRecord r;
  r.a = make_float4(v.m2.x, v.m2.y, -0.5f * RN_LOG2E * v.co.x, -RN_LOG2E * v.co.y);
  r.b = make_float4(-0.5f * RN_LOG2E * v.co.z, rn_lg2(v.co.w), v.m, 1.f / v.co.w);
  r.c = make_float4(v.r, v.g, v.b, 0.f);
  return r;
}

// Largest e over the pixel rectangle [X0, X0+15] x [Y0, Y0+7] (e is a concave quadratic in d; its
// maximum over a box whose interior misses the centre lies on an edge next to the centre).
__device__ __forceinline__ float rn_max_e_over_strip(const float4& ra, const float4& rb, float X0, float Y0) {
  const float A2 = ra.z, B2 = ra.w, C2 = rb.x, lo = rb.y;
  const float dxlo = ra.x - (X0 + 15.f), dxhi = ra.x - X0;
  const float dylo = ra.y - (Y0 + 7.f), dyhi = ra.y - Y0;
  const float dxc = fminf(fmaxf(0.f, dxlo), dxhi), dyc = fminf(fmaxf(0.f, dylo), dyhi);
  // edge dx = dxc: best dy
  const float dy1 = fminf(fmaxf(__fdividef(-B2 * dxc, 2.f * C2), dylo), dyhi);
  const float e1 = lo + A2 * dxc * dxc + B2 * dxc * dy1 + C2 * dy1 * dy1;
  // edge dy = dyc: best dx
  const float dx2 = fminf(fmaxf(__fdividef(-B2 * dyc, 2.f * A2), dxlo), dxhi);
  const float e2 = lo + A2 * dx2 * dx2 + B2 * dx2 * dyc + C2 * dyc * dyc;
  return fmaxf(e1, e2);
}

// e = log2(alpha) at the four pixels of a quad (k = 2*row + col).  Explicit rounding intrinsics: the
// forward and the backward kernel must take bit-identical alpha-filter decisions, so the compiler
// is not allowed to contract or reassociate this differently in the two kernels.
__device__ __forceinline__ void rn_eval_quad(const float4& ra, const float4& rb, float fx0, float fx1, float fy0,
                                             float fy1, float* dx, float* dy, float* e) {
  dx[0] = __fsub_rn(ra.x, fx0);
  dx[1] = __fsub_rn(ra.x, fx1);
  dy[0] = __fsub_rn(ra.y, fy0);
  dy[1] = __fsub_rn(ra.y, fy1);
  const float adx0 = __fmul_rn(ra.z, dx[0]), adx1 = __fmul_rn(ra.z, dx[1]);
  const float cyp0 = __fmaf_rn(__fmul_rn(rb.x, dy[0]), dy[0], rb.y);
  const float cyp1 = __fmaf_rn(__fmul_rn(rb.x, dy[1]), dy[1], rb.y);
  e[0] = __fmaf_rn(dx[0], __fmaf_rn(ra.w, dy[0], adx0), cyp0);
  e[1] = __fmaf_rn(dx[1], __fmaf_rn(ra.w, dy[0], adx1), cyp0);
  e[2] = __fmaf_rn(dx[0], __fmaf_rn(ra.w, dy[1], adx0), cyp1);
  e[3] = __fmaf_rn(dx[1], __fmaf_rn(ra.w, dy[1], adx1), cyp1);
}

// The alpha filter on the exponent: power > 0 (e > lo) or alpha < 1/255 => the pair is skipped.
__device__ __forceinline__ uint32_t rn_filter_quad(const float* e, float lo) {
  uint32_t pass = 0;
#pragma unroll
  for (int k = 0; k < 4; k++)
    if (e[k] <= lo && e[k] >= RN_LOG2_ALPHA_MIN) pass |= 1u << k;
  return pass;
}
