// render_common.cuh -- pieces shared by the forward and backward blend kernels.
//
// Geometry: one block per 16x16 tile, 64 threads = 2 warps that never synchronise with
// each other.  A warp owns a 16x8 pixel strip, seen as four 8x4 SUB-BLOCKS (k = 2*by + bx); a lane owns
// one pixel of each sub-block, at the same offset (lane & 7, lane >> 3).  A splat that is small against
// the strip then activates one or two sub-blocks, whose 32 pixels are exactly the 32 lanes, instead of a
// few lanes of every instruction.  The two sub-blocks of a column (bx) form a PAIR -- an 8x8 block whose
// pixels (x, y) and (x, y + 4) belong to the same lane -- and all per-pixel arithmetic is done on pairs with
// the packed FP32 instructions of sm_100 (fma/mul/add.f32x2: two lanes' worth of FMA per issue slot; both
// kernels are issue-bound, not FMA-pipe-bound).
//
// Each warp stages its tile's list itself, 32 entries at a time (lane j fetches entry j): ids two
// batches ahead in a register, attributes one batch ahead by cp.async into shared memory (no registers
// held across the blend loop), the current batch as 64-byte records in shared memory.  While a lane still
// holds its entry in registers it computes a 4-bit mask of the sub-blocks the entry can reach (exact maximum
// of the concave exponent over each 8x4 box); entries that reach no live sub-block are dropped by a ballot,
// the others are walked in list order.
//
// Record: the exponent in the log2 domain, EXPANDED ABOUT THE CENTRE OF THE STRIP.  With l = pixel - strip
// centre (|lx| <= 7.5, |ly| <= 3.5), D0 = mean2d - strip centre, d = D0 - l:
//     log2(alpha) = e(l) = lo + A2 dx^2 + B2 dx dy + C2 dy^2                          (A2 = -log2(e)/2 A, ...; lo = log2 o)
//                        = e0 + gx lx + gy ly + A2 lx^2 + B2 lx ly + C2 ly^2,
//     e0 = e at the strip centre, (gx, gy) = -(2 A2 D0x + B2 D0y, B2 D0x + 2 C2 D0y).
// e0 and g are formed in fp64 from the fp32 splat (once per entry and strip), everything per pixel is fp32.
// Why not evaluate A2 dx^2 + ... directly: for a long thin splat seen far from its centre the three terms reach
// 1e4..1e6 and cancel to O(1), so fp32 loses 1e-2..1e-1 of alpha there; about the strip centre no term of a
// contributing entry exceeds a few hundred.  The alpha filter of the method (power > 0 or alpha < 1/255 => skip)
// becomes two compares on e BEFORE any exponential is taken.
#pragma once
#include "mg_common.cuh"

#define RN_THREADS 64
#define RN_WARPS (RN_THREADS / 32)
#define RN_LOG2E 1.4426950408889634
#define RN_LN2 0.6931471805599453f
#define RN_LOG2_ALPHA_MIN -7.994353436858858f  // log2(1/255)
// The sub-block cull computes the largest e over a box along another arithmetic path than rn_eval_pair, so it keeps
// every entry within this distance (log2 units) of the threshold.
#define RN_CULL_SLACK 2e-3f
// "power > 0 => skip" cannot happen for a positive definite conic except by rounding at a pixel that coincides with the
// centre; a pair is skipped on that ground only if e exceeds lo by more than this (a conic that is not positive definite
// in its fp32 storage), and alpha never exceeds o.
#define RN_PD_SLACK 1e-3f

struct RnRecord {
  float4 a;  // e0, gx, gy, A2
  float4 b;  // B2, C2, hi = lo + RN_PD_SLACK, cap = min(0.99, o)
  float4 c;  // r, g, b, M
  float4 d;  // sub-block mask (bits), D0x, D0y, 1/o
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

// packed FP32 (sm_100): one instruction, two independent IEEE operations
__device__ __forceinline__ float2 rn_splat(float s) { return make_float2(s, s); }
__device__ __forceinline__ float2 rn_fma2(float2 a, float2 b, float2 c) { return __ffma2_rn(a, b, c); }
__device__ __forceinline__ float2 rn_mul2(float2 a, float2 b) { return __fmul2_rn(a, b); }
__device__ __forceinline__ float2 rn_add2(float2 a, float2 b) { return __fadd2_rn(a, b); }

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

// The same without the mask (the forward kernel has it already when it gathers the attributes).
__device__ __forceinline__ void rn_stage_issue_attr(RnStage* s, int lane, uint32_t id, const float2* __restrict__ means2d,
                                                    const float4* __restrict__ conic_opacity, const float* __restrict__ rgb) {
  rn_cp_async(&s->co[lane], conic_opacity + id, 16);
  rn_cp_async(&s->m2[lane], means2d + id, 8);
  rn_cp_async(&s->rgb[lane][0], rgb + 3 * (size_t)id, 4);
  rn_cp_async(&s->rgb[lane][1], rgb + 3 * (size_t)id + 1, 4);
  rn_cp_async(&s->rgb[lane][2], rgb + 3 * (size_t)id + 2, 4);
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

// The record of an entry for the strip whose centre is (Xc, Yc).  e0 and g in fp64: the expansion point is up to
// thousands of pixels from the splat's centre and e0 is what remains of terms of that size squared.
#ifndef RN_STAGE_T
#define RN_STAGE_T double  // (-DRN_STAGE_T=float: to measure what the fp64 staging costs; loses the accuracy it is there for)
#endif
__device__ __forceinline__ RnRecord rn_make_record(const RnRaw& v, float Xc, float Yc) {
  typedef RN_STAGE_T D;
  const D D0x = (D)v.m2.x - (D)Xc, D0y = (D)v.m2.y - (D)Yc;  // exact in fp64
  const D A2 = (D)(-0.5 * RN_LOG2E) * (D)v.co.x, B2 = (D)(-RN_LOG2E) * (D)v.co.y, C2 = (D)(-0.5 * RN_LOG2E) * (D)v.co.z;
  const float lo = rn_lg2(v.co.w);
  const D hx = A2 * D0x, hy = C2 * D0y;
  const D e0 = (D)lo + (hx + B2 * D0y) * D0x + hy * D0y;
  const D gx = -((D)2 * hx + B2 * D0y), gy = -(B2 * D0x + (D)2 * hy);
  RnRecord r;
  r.a = make_float4((float)e0, (float)gx, (float)gy, (float)A2);
  r.b = make_float4((float)B2, (float)C2, lo + RN_PD_SLACK, fminf(MG_ALPHA_MAX, v.co.w));
  r.c = make_float4(v.r, v.g, v.b, v.m);
  r.d = make_float4(0.f, (float)D0x, (float)D0y, 1.f / v.co.w);
  return r;
}

// Bit k set = the entry can pass the alpha filter somewhere in sub-block k of the strip.  In the strip's local
// coordinates the boxes are [xlo, xhi] x [ylo, yhi] with x-intervals [-7.5, -0.5], [0.5, 7.5] and y-intervals
// [-3.5, -0.5], [0.5, 3.5].  e is a concave quadratic with its maximum at the splat's centre c = D0.  If c lies outside
// a box, the maximum over the box lies on an edge FACING c (moving from the maximiser towards c increases e, so that
// direction leaves the box): the edge lx = clamp(cx) with the best ly, or the edge ly = clamp(cy) with the best lx.  (If
// c is inside the box's range along an axis, that candidate is an interior line: harmless.)  The four boxes share their
// two x-intervals and two y-intervals, so everything that depends on one axis is computed twice, not four times.
__device__ __forceinline__ uint32_t rn_subblock_mask(const RnRecord& r) {
  const float e0 = r.a.x, gx = r.a.y, gy = r.a.z, A2 = r.a.w, B2 = r.b.x, C2 = r.b.y;
  const float cx = r.d.y, cy = r.d.z;
  const float inv2C = __fdividef(-0.5f, C2), inv2A = __fdividef(-0.5f, A2);
  const float xlo[2] = {-7.5f, 0.5f}, xhi[2] = {-0.5f, 7.5f}, ylo[2] = {-3.5f, 0.5f}, yhi[2] = {-0.5f, 3.5f};
  float qx[2], sy[2], ty[2], qy[2], sx[2], tx[2];
#pragma unroll
  for (int i = 0; i < 2; i++) {
    const float lxc = fminf(fmaxf(cx, xlo[i]), xhi[i]);
    qx[i] = fmaf(lxc, fmaf(A2, lxc, gx), e0);  // e on the line lx = lxc at ly = 0
    sy[i] = fmaf(B2, lxc, gy);                 // its slope in ly there
    ty[i] = sy[i] * inv2C;                     // best ly on that line, before clamping
    const float lyc = fminf(fmaxf(cy, ylo[i]), yhi[i]);
    qy[i] = fmaf(lyc, fmaf(C2, lyc, gy), e0);
    sx[i] = fmaf(B2, lyc, gx);
    tx[i] = sx[i] * inv2A;
  }
  uint32_t m = 0;
#pragma unroll
  for (int k = 0; k < 4; k++) {
    const int ix = k & 1, iy = k >> 1;
    const float ly1 = fminf(fmaxf(ty[ix], ylo[iy]), yhi[iy]);
    const float e1 = fmaf(ly1, fmaf(C2, ly1, sy[ix]), qx[ix]);
    const float lx2 = fminf(fmaxf(tx[iy], xlo[ix]), xhi[ix]);
    const float e2 = fmaf(lx2, fmaf(A2, lx2, sx[iy]), qy[iy]);
    if (fmaxf(e1, e2) >= RN_LOG2_ALPHA_MIN - RN_CULL_SLACK) m |= 1u << k;
  }
  return m;
}

// A lane's pixels in the strip's local coordinates: columns lx.x (bx = 0), lx.y (bx = 1); rows ly.x (by = 0), ly.y (by = 1).
struct RnLane {
  float2 lx, ly;
};
__device__ __forceinline__ RnLane rn_lane(int lane) {
  RnLane L;
  L.lx = make_float2((float)(lane & 7) - 7.5f, (float)(lane & 7) + 0.5f);
  L.ly = make_float2((float)(lane >> 3) - 3.5f, (float)(lane >> 3) + 0.5f);
  return L;
}

// Per-entry partial terms of e for a lane's two columns and two rows (5 packed instructions).
// Explicit IEEE intrinsics throughout: the forward and the backward kernel must take bit-identical alpha-filter
// decisions, so the compiler may not contract or reassociate this differently in the two kernels.
struct RnPartial {
  float2 col;  // lx (gx + A2 lx)      per column
  float2 bl;   // B2 lx                per column
  float2 row;  // e0 + ly (gy + C2 ly) per row
};
__device__ __forceinline__ RnPartial rn_partial(const float4& ra, const float4& rb, const RnLane& L) {
  RnPartial p;
  p.col = rn_mul2(rn_fma2(rn_splat(ra.w), L.lx, rn_splat(ra.y)), L.lx);
  p.bl = rn_mul2(rn_splat(rb.x), L.lx);
  p.row = rn_fma2(rn_fma2(rn_splat(rb.y), L.ly, rn_splat(ra.z)), L.ly, rn_splat(ra.x));
  return p;
}

// e = log2(alpha) at the lane's two pixels of column c (.x: row by = 0, sub-block c; .y: row by = 1, sub-block c + 2).
__device__ __forceinline__ float2 rn_eval_pair(const RnPartial& p, const RnLane& L, int c) {
  const float col = c ? p.col.y : p.col.x, bl = c ? p.bl.y : p.bl.x;
  return rn_fma2(rn_splat(bl), L.ly, rn_add2(p.row, rn_splat(col)));
}

// The alpha filter on the exponent: power > 0 (beyond rounding: e > hi) or alpha < 1/255 => the pair is skipped.
__device__ __forceinline__ bool rn_filter(float e, float hi) { return e <= hi && e >= RN_LOG2_ALPHA_MIN; }
