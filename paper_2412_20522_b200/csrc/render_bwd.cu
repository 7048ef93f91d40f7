// render_bwd.cu -- mg_render_bwd: reverse traversal of a tile's list (step a8).
// Per pixel, from its last contributor back to the front:
//   T_i      = T_{i+1} / (1 - M_i alpha_i)                       (Eq. 16 taken apart one factor at a time)
//   b_i      = M_i alpha_i c_i + (1 - M_i alpha_i) b_{i+1}        (Eq. 11), b_{N+1} = 0
//   X_i      = T_i g.(c_i - b_{i+1}) - T_{N+1}/(1 - M_i alpha_i) g.c_bg,   g = dL/dc(x)
//   dL/dM_i += alpha_i X_i                                        (Eq. 18)
//   dL/dalpha_i = M_i X_i ;  dL/dc_i += M_i alpha_i T_i g
// Only the scalar g.b is carried (g is fixed per pixel), not the colour b itself.
// With q = alpha_i dL/dalpha_i (zero where the 0.99 clamp is active), the sums over pixels of
// q, q dx, q dy, q dx^2, q dx dy, q dy^2 give dL/d(opacity, centre, conic) by a per-entry linear map.
//
// FP32-issue and shuffle bound.  Same geometry, staging, records (expanded about the strip centre), sub-block cull and
// packed evaluation of the exponent as the forward kernel (render_common.cuh), walking each warp's strip from its
// largest n_contrib back to the front.  The blend sections are per sub-block and scalar: packed over the two
// sub-blocks of a column they ran for both whenever either was reached (measured: 1.01 ms against 0.88 ms).
//  * An entry with M = 0 leaves T and b unchanged and receives dL/dM only (Fig. 1): a
//    warp-uniform branch with a third of the arithmetic, one plain butterfly and one atomic.
//  * Otherwise a lane sums its (up to 4) pixels in registers; the 10 per-entry sums are reduced over
//    the warp by a transposing butterfly (12 shuffles instead of 50) that leaves sum s in lane pair s,
//    and 10 lanes issue one red.global.add each.
#include "render_common.cuh"

#ifndef RN_BWD_MINB
#define RN_BWD_MINB 11  // minimum resident blocks per SM asked of ptxas (register budget)
#endif

namespace {

struct BwdTargets {
  float* base[10];
  int stride[10];
  int offset[10];
};

// Sum each of 10 per-lane values over the 32 lanes.  Returns, in lanes whose slot (see slot_of_lane)
// is s >= 0, the total of v[s].
__device__ __forceinline__ float transpose_reduce10(const float* v, int lane) {
  const bool b4 = lane & 16, b3 = lane & 8, b2 = lane & 4, b1 = lane & 2;
  float u[5];
#pragma unroll
  for (int i = 0; i < 5; i++) {
    const float send = b4 ? v[i] : v[i + 5];
    const float keep = b4 ? v[i + 5] : v[i];
    u[i] = keep + __shfl_xor_sync(0xffffffffu, send, 16);
  }
  // b3 = 0 keeps (u0,u1,u2), b3 = 1 keeps (u3,u4,-)
  float w0, w1, w2;
  {
    const float r0 = __shfl_xor_sync(0xffffffffu, b3 ? u[0] : u[3], 8);
    const float r1 = __shfl_xor_sync(0xffffffffu, b3 ? u[1] : u[4], 8);
    const float r2 = __shfl_xor_sync(0xffffffffu, b3 ? u[2] : 0.f, 8);
    w0 = (b3 ? u[3] : u[0]) + r0;
    w1 = (b3 ? u[4] : u[1]) + r1;
    w2 = (b3 ? 0.f : u[2]) + r2;
  }
  // b2 = 0 keeps (w0,w1), b2 = 1 keeps (w2,-)
  float x0, x1;
  {
    const float r0 = __shfl_xor_sync(0xffffffffu, b2 ? w0 : w2, 4);
    const float r1 = __shfl_xor_sync(0xffffffffu, b2 ? w1 : 0.f, 4);
    x0 = (b2 ? w2 : w0) + r0;
    x1 = (b2 ? 0.f : w1) + r1;
  }
  // b1 = 0 keeps x0, b1 = 1 keeps x1
  float y = (b1 ? x1 : x0) + __shfl_xor_sync(0xffffffffu, b1 ? x0 : x1, 2);
  y += __shfl_xor_sync(0xffffffffu, y, 1);
  return y;
}

// Which of the 10 sums a lane holds after transpose_reduce10 (-1: none, or the odd twin of a pair).
__device__ __forceinline__ int slot_of_lane(int lane) {
  if (lane & 1) return -1;
  const int b4 = (lane >> 4) & 1, b3 = (lane >> 3) & 1, b2 = (lane >> 2) & 1, b1 = (lane >> 1) & 1;
  int idx;
  if (!b3) idx = b2 ? (b1 ? -1 : 2) : b1;
  else idx = b2 ? -1 : 3 + b1;
  return idx < 0 ? -1 : 5 * b4 + idx;
}

__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
  for (int o = 16; o >= 1; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

template <bool kBg>
__global__ void __launch_bounds__(RN_THREADS, RN_BWD_MINB) render_bwd_kernel(
    int W, int H, int gw, float bg0, float bg1, float bg2, const uint32_t* __restrict__ sorted_ids,
    const uint2* __restrict__ tile_ranges, const uint32_t* __restrict__ tile_order,
    const float2* __restrict__ means2d, const float4* __restrict__ conic_opacity, const float* __restrict__ rgb,
    const float* __restrict__ masks, const float* __restrict__ final_T, const uint32_t* __restrict__ n_contrib, const float* __restrict__ dL_dimage,
    BwdTargets tg) {
  __shared__ RnRecord buf_all[RN_WARPS][32];
  __shared__ RnStage stage_all[RN_WARPS];
  __shared__ uint32_t ids_all[RN_WARPS][32];
  const int tile = tile_order ? (int)tile_order[blockIdx.x] : (int)blockIdx.x;  // longest lists first
  const int tx = tile % gw, ty = tile / gw;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  RnRecord* buf = buf_all[warp];
  RnStage* stage = &stage_all[warp];
  uint32_t* ids_sh = ids_all[warp];
  const uint2 range = tile_ranges[tile];
  const uint32_t* ids = sorted_ids + range.x;

  // pixels of this lane: (px[c], py[r]); sub-block k = c + 2 r; pair c = the sub-blocks k = c and k = c + 2
  const int X0i = tx * MG_TILE, Y0i = ty * MG_TILE + 8 * warp;
  const int px[2] = {X0i + (lane & 7), X0i + 8 + (lane & 7)};
  const int py[2] = {Y0i + (lane >> 3), Y0i + 4 + (lane >> 3)};
  const float Xc = (float)X0i + 7.5f, Yc = (float)Y0i + 3.5f;  // centre of the strip: origin of the records
  const RnLane L = rn_lane(lane);

  // per-pixel state
  float T[4], gB[4], g0[4], g1[4], g2[4], tfg[4];
  uint32_t last[4], sbmax[4];
  const size_t plane = (size_t)W * H;
  uint32_t wmax = 0;
#pragma unroll
  for (int k = 0; k < 4; k++) {
    const int x = px[k & 1], y = py[k >> 1];
    T[k] = 1.f; gB[k] = 0.f; g0[k] = g1[k] = g2[k] = 0.f; tfg[k] = 0.f; last[k] = 0;
    if (x < W && y < H) {
      const size_t pix = (size_t)y * W + x;
      T[k] = final_T[pix];
      last[k] = n_contrib[pix];
      g0[k] = dL_dimage[pix];
      g1[k] = dL_dimage[plane + pix];
      g2[k] = dL_dimage[2 * plane + pix];
      if (kBg) tfg[k] = T[k] * (g0[k] * bg0 + g1[k] * bg1 + g2[k] * bg2);  // T_{N+1} g.c_bg
    }
    sbmax[k] = __reduce_max_sync(0xffffffffu, last[k]);  // warp-uniform: last contributor of sub-block k
    wmax = max(wmax, sbmax[k]);
  }
  wmax = min(wmax, range.y - range.x);  // never walk past the tile's own list
  if (wmax == 0) return;                // warps do not synchronise with each other

  // where this lane's reduced sum goes
  const int slot = slot_of_lane(lane);
  float* tgt_ptr = nullptr;  // element 0 of this lane's component; Gaussian id lives tgt_stride floats further on
  uint32_t tgt_stride = 0;
#pragma unroll
  for (int s = 0; s < 10; s++)
    if (slot == s) { tgt_ptr = tg.base[s] + tg.offset[s]; tgt_stride = (uint32_t)tg.stride[s]; }
  float* const dmask = tg.base[9];

  const int n = (int)wmax;  // entries at positions > wmax are never visited by this warp
  const int bstart = ((n - 1) >> 5) << 5;
  // prologue: gather of the last batch in flight, ids of the one before it in a register
  uint32_t id_cur = bstart + lane < n ? ids[bstart + lane] : 0u;
  if (bstart + lane < n) rn_stage_issue(stage, lane, id_cur, means2d, conic_opacity, rgb, masks);
  rn_cp_async_commit();
  uint32_t id_nxt = bstart >= 32 ? ids[bstart - 32 + lane] : 0u;

  for (int base = bstart; base >= 0; base -= 32) {
    rn_cp_async_wait_all();  // this lane's entry of the current batch has landed
    __syncwarp();            // every lane is done reading the previous batch's records
    uint32_t m4 = 0;
    if (base + lane < n) {
      RnRecord rec = rn_make_record(rn_stage_read(stage, lane), Xc, Yc);
      m4 = rn_subblock_mask(rec);
      const uint32_t mypos = (uint32_t)(base + lane + 1);
#pragma unroll
      for (int k = 0; k < 4; k++)
        if (mypos > sbmax[k]) m4 &= ~(1u << k);
      rec.d.x = __uint_as_float(m4);
      if (m4) {
        buf[lane] = rec;
        ids_sh[lane] = id_cur;
      }
    }
    // gather of the next batch (towards the front) and id load of the one after
    if (base >= 32) rn_stage_issue(stage, lane, id_nxt, means2d, conic_opacity, rgb, masks);
    rn_cp_async_commit();
    id_cur = id_nxt;
    id_nxt = base >= 64 ? ids[base - 64 + lane] : 0u;
    __syncwarp();  // records visible to the whole warp
    uint32_t todo = __ballot_sync(0xffffffffu, m4 != 0);
    while (todo) {
      const int jj = 31 - __clz(todo);
      todo &= ~(1u << jj);
      const float4 ra = buf[jj].a, rb = buf[jj].b, rc = buf[jj].c, rd = buf[jj].d;
      // the same record is read by every lane: a warp reduction hands the compiler that fact (uniform registers and
      // branches for everything that depends on the sub-block mask and on M)
      const uint32_t sb = __reduce_or_sync(0xffffffffu, __float_as_uint(rd.x));
      const float hi = rb.z, cap = rb.w;
      const float m = __uint_as_float(__reduce_or_sync(0xffffffffu, __float_as_uint(rc.w)));
      const uint32_t pos = (uint32_t)(base + jj + 1);
      const RnPartial p = rn_partial(ra, rb, L);

      // e at the lane's four pixels: two packed evaluations
      float ek[4];
      {
        const float2 ea = rn_eval_pair(p, L, 0), eb = rn_eval_pair(p, L, 1);
        ek[0] = ea.x; ek[2] = ea.y; ek[1] = eb.x; ek[3] = eb.y;
      }
      if (m == 0.f) {
        // masked entry: a = 0, T_i = T_{i+1}, b unchanged; only dL/dM = sum alpha X (Eq. 18)
        float dm = 0.f;
#pragma unroll
        for (int k = 0; k < 4; k++) {
          if ((sb >> k) & 1u) {
            // branch-free: a pixel that fails the filter gets alpha = 0 and adds nothing
            const bool pass = rn_filter(ek[k], hi) && pos <= last[k];
            const float alpha = pass ? fminf(cap, rn_ex2(ek[k])) : 0.f;
            const float gc = g0[k] * rc.x + g1[k] * rc.y + g2[k] * rc.z;
            const float X = kBg ? T[k] * (gc - gB[k]) - tfg[k] : T[k] * (gc - gB[k]);
            dm = fmaf(alpha, X, dm);
          }
        }
        if (__any_sync(0xffffffffu, dm != 0.f)) {
          const float total = warp_sum(dm);
          if (lane == 0) atomicAdd(dmask + ids_sh[jj], total);
        }
        continue;
      }
      float S = 0.f, Sx = 0.f, Sy = 0.f, Sxx = 0.f, Sxy = 0.f, Syy = 0.f;
      float dr = 0.f, dg = 0.f, db = 0.f, dm = 0.f;
      bool contrib = false;
#pragma unroll
      for (int k = 0; k < 4; k++) {
        if ((sb >> k) & 1u) {
          const bool pass = rn_filter(ek[k], hi) && pos <= last[k];
          if (__any_sync(0xffffffffu, pass)) {
            contrib = true;
            // branch-free inside the section: a lane whose pixel fails the filter blends with alpha = 0, which adds
            // nothing to any sum; its T and g.b are kept by a select
            const float raw_alpha = rn_ex2(ek[k]);
            const float alpha = pass ? fminf(cap, raw_alpha) : 0.f;
            const float a = m * alpha;
            const float oma = 1.f - a;
            const float inv = rn_rcp(oma);
            const float Ti = T[k] * inv;
            const float gc = g0[k] * rc.x + g1[k] * rc.y + g2[k] * rc.z;
            const float X = kBg ? Ti * (gc - gB[k]) - tfg[k] * inv : Ti * (gc - gB[k]);
            dm = fmaf(alpha, X, dm);
            const float wgt = a * Ti;
            dr = fmaf(wgt, g0[k], dr);
            dg = fmaf(wgt, g1[k], dg);
            db = fmaf(wgt, g2[k], db);
            gB[k] = pass ? fmaf(a, gc, oma * gB[k]) : gB[k];
            T[k] = pass ? Ti : T[k];
            const float q = raw_alpha <= MG_ALPHA_MAX ? alpha * (m * X) : 0.f;  // no gradient through the active clamp
            const float ddx = rd.y - ((k & 1) ? L.lx.y : L.lx.x), ddy = rd.z - ((k >> 1) ? L.ly.y : L.ly.x);  // d = D0 - l
            const float qx = q * ddx, qy = q * ddy;
            S += q; Sx += qx; Sy += qy;
            Sxx = fmaf(qx, ddx, Sxx);
            Sxy = fmaf(qx, ddy, Sxy);
            Syy = fmaf(qy, ddy, Syy);
          }
        }
      }
      if (!contrib) continue;
      // per-entry linear map: true conic (A,B,C) = (-2 ln2 A2, -ln2 B2, -2 ln2 C2)
      float v[10];
      v[0] = RN_LN2 * (2.f * ra.w * Sx + rb.x * Sy);   // dL/dmean2d.x = -(A Sx + B Sy)
      v[1] = RN_LN2 * (rb.x * Sx + 2.f * rb.y * Sy);   // dL/dmean2d.y = -(B Sx + C Sy)
      v[2] = -0.5f * Sxx;                              // dL/dA
      v[3] = -Sxy;                                     // dL/dB
      v[4] = -0.5f * Syy;                              // dL/dC
      v[5] = S * rd.w;                                 // dL/do = sum q / o
      v[6] = dr; v[7] = dg; v[8] = db;
      v[9] = dm;
      const float total = transpose_reduce10(v, lane);
      if (slot >= 0 && total != 0.f) {
        const uint32_t id = ids_sh[jj];
        atomicAdd(tgt_ptr + (size_t)id * tgt_stride, total);
      }
    }
  }
}

}  // namespace

extern "C" int mg_render_bwd(const mg_camera* cam, int64_t N, const uint32_t* sorted_ids, const uint32_t* tile_ranges,
                             const uint32_t* tile_order, const float* means2d, const float* conic_opacity, const float* rgb, const float* masks,
                             const float* final_T, const uint32_t* n_contrib, const float* dL_dimage,
                             float* dL_dmeans2d, float* dL_dconic, float* dL_dopacity, float* dL_drgb, float* dL_dmask,
                             void* stream) {
  if (int rc = mg_check_camera(cam)) return rc;
  MG_REQUIRE(N >= 0 && N < (int64_t)1 << 31, "N must be in [0, 2^31)");
  MG_REQUIRE(tile_ranges && final_T && n_contrib && dL_dimage, "null per-pixel array or tile_ranges");
  cudaStream_t st = (cudaStream_t)stream;
  if (N > 0) {
    MG_REQUIRE(means2d && conic_opacity && rgb && masks, "null splat array");
    MG_REQUIRE(dL_dmeans2d && dL_dconic && dL_dopacity && dL_drgb && dL_dmask, "null gradient array");
    MG_CHECK_CUDA(cudaMemsetAsync(dL_dmeans2d, 0, sizeof(float) * 2 * N, st));
    MG_CHECK_CUDA(cudaMemsetAsync(dL_dconic, 0, sizeof(float) * 3 * N, st));
    MG_CHECK_CUDA(cudaMemsetAsync(dL_dopacity, 0, sizeof(float) * N, st));
    MG_CHECK_CUDA(cudaMemsetAsync(dL_drgb, 0, sizeof(float) * 3 * N, st));
    MG_CHECK_CUDA(cudaMemsetAsync(dL_dmask, 0, sizeof(float) * N, st));
  }
  BwdTargets tg;
  float* bases[10] = {dL_dmeans2d, dL_dmeans2d, dL_dconic, dL_dconic, dL_dconic, dL_dopacity, dL_drgb, dL_drgb, dL_drgb, dL_dmask};
  const int strides[10] = {2, 2, 3, 3, 3, 1, 3, 3, 3, 1};
  const int offsets[10] = {0, 1, 0, 1, 2, 0, 0, 1, 2, 0};
  for (int s = 0; s < 10; s++) { tg.base[s] = bases[s]; tg.stride[s] = strides[s]; tg.offset[s] = offsets[s]; }
  const int gw = mg_grid_w(cam), gh = mg_grid_h(cam);
  // a black background (the common case) has no T_{N+1} g.c_bg term: four registers and two instructions per blend less
  const bool has_bg = cam->bg[0] != 0.f || cam->bg[1] != 0.f || cam->bg[2] != 0.f;
  if (has_bg)
    render_bwd_kernel<true><<<gw * gh, RN_THREADS, 0, st>>>(cam->width, cam->height, gw, cam->bg[0], cam->bg[1], cam->bg[2],
                                                            sorted_ids, (const uint2*)tile_ranges, tile_order, (const float2*)means2d,
                                                            (const float4*)conic_opacity, rgb, masks, final_T, n_contrib,
                                                            dL_dimage, tg);
  else
    render_bwd_kernel<false><<<gw * gh, RN_THREADS, 0, st>>>(cam->width, cam->height, gw, 0.f, 0.f, 0.f,
                                                             sorted_ids, (const uint2*)tile_ranges, tile_order, (const float2*)means2d,
                                                             (const float4*)conic_opacity, rgb, masks, final_T, n_contrib,
                                                             dL_dimage, tg);
  MG_CHECK_LAUNCH();
  return MG_OK;
}
