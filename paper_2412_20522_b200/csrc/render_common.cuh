// render_common.cuh -- pieces shared by the forward and backward blend kernels.
//
// Geometry: one block per 16x16 tile, 64 threads = 2 warps that never synchronise with
// each other.  A warp owns a 16x8 pixel strip, seen as four 8x4 SUB-BLOCKS (k = 2*by + bx); a lane owns
// one pixel of each sub-block, at the same offset (lane & 7, lane >> 3).  A splat that is small against
// the strip then activates one or two sub-blocks, whose 32 pixels are exactly the 32 lanes, instead of a
// few lanes of every instruction.
//
// Each warp stages its tile's list itself, 32 entries at a time (lane j fetches entry j): ids two
// batches ahead in a register, attributes one batch ahead by cp.async into shared memory (no registers
// held across the blend loop), the current batch as 48-byte records in shared memory.  While a lane still holds its entry in registers it computes a 4-bit mask of the
// sub-blocks the entry can reach (exact maximum of the concave exponent over each 8x4 box); entries
// that reach no live sub-block are dropped by a ballot, the others are walked in list order.
//
// Record: the conic is pre-scaled into the log2 domain and the opacity folded in as an offset, so that
//     log2(alpha) = e = lo + A2 dx^2 + B2 dx dy + C2 dy^2,   d = mean2d - pixel,
// and the alpha filter of the method (power > 0 or alpha < 1/255 => skip) becomes two compares on e
// BEFORE any exponential is taken:  e > lo  or  e < log2(1/255).
#pragma once
#include "mg_common.cuh"

#define RN_THREADS 64
#define RN_WARPS (RN_THREADS / 32)
#define RN_LOG2E 1.4426950408889634f
#define RN_LN2 0.6931471805599453f
#define RN_LOG2_ALPHA_MIN -7.994353436858858f  // log2(1/255)
// The sub-block cull computes the largest e over a box along another arithmetic path than rn_eval, so it keeps every
// entry within a slack of the threshold: 2^-10, plus 2^-21 of the largest magnitude the three quadratic terms can reach
// over the strip (for a long thin splat far from its centre they reach 1e4..1e6 and cancel: the fp32 error of e is a
// few ulps of the terms, not of e).
#define RN_CULL_SLACK 1e-3f
#define RN_CULL_SLACK_REL 4.8e-7f

struct RnRecord {
  float4 a;  // mx, my, A2, B2
  float4 b;  // C2, lo, mask, 1/o
  float4 c;  // r, g, b, sub-block mask (bits)
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
__device__ __forceinline__ float rn_rcp(float x) {
  float y;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}

struct RnRaw {  // attributes of one list entry as gathered from global memory
  float2 m2;
  float4 co;
  float r, g, b, m;
};

// Per-warp landing zone of the asynchronous gather (cp.async, LDGSTS): lane j's entry lands in slot j of
// each array, so the gather of the next batch costs no registers while the current batch is blended.
// A slot is written and read by the same lane only.
struct RnStage {
  float4 co[32];
  float2 m2[32];
  float rgb[32][3];
  float m[32];
};

__device__ __forceinline__ void rn_cp_async(void* smem_dst, const void* gmem_src, int bytes) {
  const uint32_t d = (uint32_t)__cvta_generic_to_shared(smem_dst);
  if (bytes == 16) asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gmem_src) : "memory");
  else if (bytes == 8) asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(d), "l"(gmem_src) : "memory");
  else asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(d), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void rn_cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void rn_cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

__device__ __forceinline__ void rn_stage_issue(RnStage* s, int lane, uint32_t id, const float2* __restrict__ means2d,
                                               const float4* __restrict__ conic_opacity, const float* __restrict__ rgb,
                                               const float* __restrict__ masks) {
  rn_cp_async(&s->co[lane], conic_opacity + id, 16);
  rn_cp_async(&s->m2[lane], means2d + id, 8);
  rn_cp_async(&s->rgb[lane][0], rgb + 3 * (size_t)id, 4);
  rn_cp_async(&s->rgb[lane][1], rgb + 3 * (size_t)id + 1, 4);
  rn_cp_async(&s->rgb[lane][2], rgb + 3 * (size_t)id + 2, 4);
  rn_cp_async(&s->m[lane], masks + id, 4);
}

__device__ __forceinline__ RnRaw rn_stage_read(const RnStage* s, int lane) {
  RnRaw v;
  v.m2 = s->m2[lane];
  v.co = s->co[lane];
  v.r = s->rgb[lane][0];
  v.g = s->rgb[lane][1];
  v.b = s->rgb[lane][2];
  v.m = s->m[lane];
  return v;
}

__device__ __forceinline__ RnRecord rn_make_record(const RnRaw& v) {
  RnRecord r;
  r.a = make_float4(v.m2.x, v.m2.y, -0.5f * RN_LOG2E * v.co.x, -RN_LOG2E * v.co.y);
  r.b = make_float4(-0.5f * RN_LOG2E * v.co.z, rn_lg2(v.co.w), v.m, 1.f / v.co.w);
  r.c = make_float4(v.r, v.g, v.b, 0.f);
  return r;
}

// Bit k set = the entry can pass the alpha filter somewhere in sub-block k of the strip at (X0, Y0).
// Per box: the largest e over the pixel rectangle (e is a concave quadratic in d; its maximum over a box whose
// interior misses the centre lies on an edge next to the centre: the edge dx = dxc with the best dy, or the edge
// dy = dyc with the best dx).  The four 8x4 boxes share their two x-intervals and two y-intervals, so everything that
// depends on one axis only (clamped offsets, the unconstrained optimum along the other axis, the pure quadratic
// terms) is computed twice, not four times; per box only the two clamps and the two edge values remain.
__device__ __forceinline__ uint32_t rn_subblock_mask(const float4& ra, const float4& rb, float X0, float Y0) {
  const float A2 = ra.z, B2 = ra.w, C2 = rb.x, lo = rb.y;
  const float inv2C = __fdividef(1.f, 2.f * C2), inv2A = __fdividef(1.f, 2.f * A2);
  float dxlo[2], dxhi[2], dxc[2], ty[2], qx[2], bx[2];  // per x-interval
  float dylo[2], dyhi[2], dyc[2], tx[2], qy[2], by[2];  // per y-interval
#pragma unroll
  for (int i = 0; i < 2; i++) {
    dxlo[i] = ra.x - (X0 + 8.f * i + 7.f); dxhi[i] = ra.x - (X0 + 8.f * i);
    dxc[i] = fminf(fmaxf(0.f, dxlo[i]), dxhi[i]);
    ty[i] = -B2 * dxc[i] * inv2C;       // best dy on the edge dx = dxc, before clamping
    qx[i] = lo + A2 * dxc[i] * dxc[i];  // lo + A2 dxc^2
    bx[i] = B2 * dxc[i];
    dylo[i] = ra.y - (Y0 + 4.f * i + 3.f); dyhi[i] = ra.y - (Y0 + 4.f * i);
    dyc[i] = fminf(fmaxf(0.f, dylo[i]), dyhi[i]);
    tx[i] = -B2 * dyc[i] * inv2A;
    qy[i] = lo + C2 * dyc[i] * dyc[i];
    by[i] = B2 * dyc[i];
  }
  // largest |dx|, |dy| over the strip -> bound of the magnitude of the terms of e at any of its pixels
  const float Dx = fmaxf(fabsf(dxlo[1]), fabsf(dxhi[0])), Dy = fmaxf(fabsf(dylo[1]), fabsf(dyhi[0]));
  const float mag = fabsf(A2) * Dx * Dx + fabsf(B2) * Dx * Dy + fabsf(C2) * Dy * Dy + fabsf(lo);
  const float thresh = RN_LOG2_ALPHA_MIN - RN_CULL_SLACK - RN_CULL_SLACK_REL * mag;
  uint32_t m = 0;
#pragma unroll
  for (int k = 0; k < 4; k++) {
    const int ix = k & 1, iy = k >> 1;
    const float dy1 = fminf(fmaxf(ty[ix], dylo[iy]), dyhi[iy]);
    const float e1 = qx[ix] + (bx[ix] + C2 * dy1) * dy1;
    const float dx2 = fminf(fmaxf(tx[iy], dxlo[ix]), dxhi[ix]);
    const float e2 = qy[iy] + (by[iy] + A2 * dx2) * dx2;
    if (fmaxf(e1, e2) >= thresh) m |= 1u << k;
  }
  return m;
}

// Per-entry partial products of e for a lane's pixel columns (bx = 0, 1) and rows (by = 0, 1).
struct RnPartial {
  float dx[2], dy[2], adx[2], cyp[2];
};

// Explicit rounding intrinsics: the forward and the backward kernel must take bit-identical
// alpha-filter decisions, so the compiler is not allowed to contract or reassociate this differently
// in the two kernels.
__device__ __forceinline__ RnPartial rn_partial(const float4& ra, const float4& rb, const float* fx, const float* fy) {
  RnPartial p;
#pragma unroll
  for (int i = 0; i < 2; i++) {
    p.dx[i] = __fsub_rn(ra.x, fx[i]);
    p.dy[i] = __fsub_rn(ra.y, fy[i]);
    p.adx[i] = __fmul_rn(ra.z, p.dx[i]);
    p.cyp[i] = __fmaf_rn(__fmul_rn(rb.x, p.dy[i]), p.dy[i], rb.y);
  }
  return p;
}

// e = log2(alpha) at the lane's pixel of sub-block k.
__device__ __forceinline__ float rn_eval(const RnPartial& p, float B2, int k) {
  return __fmaf_rn(p.dx[k & 1], __fmaf_rn(B2, p.dy[k >> 1], p.adx[k & 1]), p.cyp[k >> 1]);
}

// The alpha filter on the exponent: power > 0 (e > lo) or alpha < 1/255 => the pair is skipped.
__device__ __forceinline__ bool rn_filter(float e, float lo) { return e <= lo && e >= RN_LOG2_ALPHA_MIN; }
