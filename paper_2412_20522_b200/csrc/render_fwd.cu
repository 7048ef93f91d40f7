// render_fwd.cu -- mg_render_fwd: masked front-to-back blend of a 16x16 tile (step a7).
// Eq. 3-4: C += M_i alpha_i T_i c_i,  T_{i+1} = (1 - M_i alpha_i) T_i;
// Eq. 9-10: image = C + T_{N+1} c_bg.  Thresholds: DESIGN.md readings 1-5.
//
// FP32-issue bound (no dense contraction on this path, so no tensor cores).  Design (render_common.cuh):
//  * 2 independent warps per tile, each a 16x8 strip of four 8x4 sub-blocks, one pixel of each per lane;
//  * per warp, 32 list entries at a time: attributes gathered one batch ahead (cp.async), the record of the entry
//    expanded about the strip's centre and a 4-bit sub-block reach mask per entry (lanes = entries), a ballot, then the
//    surviving entries in list order;
//  * per surviving entry only the reachable, still-live pairs of sub-blocks are evaluated, two pixels per packed
//    FP32 instruction; the alpha filter is two compares on the exponent, the exponential is taken only for pixels
//    that pass;
//  * an entry with M = 0 changes neither C nor T and cannot stop a pixel, and n_contrib counts
//    the entries consumed before the stop (include/mg.h, reading 5), so masked entries are dropped when the
//    batch is staged: the forward pass costs nothing for them;
//  * a warp leaves when all its pixels have stopped.
#include "render_common.cuh"

#ifndef RN_FWD_MINB
#define RN_FWD_MINB 14  // minimum resident blocks per SM asked of ptxas (register budget)
#endif

namespace {

__global__ void __launch_bounds__(RN_THREADS, RN_FWD_MINB) render_fwd_kernel(
    int W, int H, int gw, float bg0, float bg1, float bg2, const uint32_t* __restrict__ sorted_ids,
    const uint2* __restrict__ tile_ranges, const uint32_t* __restrict__ tile_order,
    const float2* __restrict__ means2d, const float4* __restrict__ conic_opacity, const float* __restrict__ rgb,
    const float* __restrict__ masks, float* __restrict__ image, float* __restrict__ final_T, uint32_t* __restrict__ n_contrib) {
  __shared__ RnRecord buf_all[RN_WARPS][32];
  __shared__ RnStage stage_all[RN_WARPS];
  const int tile = tile_order ? (int)tile_order[blockIdx.x] : (int)blockIdx.x;  // longest lists first
  const int tx = tile % gw, ty = tile / gw;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  RnRecord* buf = buf_all[warp];
  RnStage* stage = &stage_all[warp];
  const uint2 range = tile_ranges[tile];
  const int n = (int)(range.y - range.x);
  const uint32_t* ids = sorted_ids + range.x;

  // pixels of this lane: (px[c], py[r]); sub-block k = c + 2 r; pair c = the sub-blocks k = c and k = c + 2
  const int X0i = tx * MG_TILE, Y0i = ty * MG_TILE + 8 * warp;
  const int px[2] = {X0i + (lane & 7), X0i + 8 + (lane & 7)};
  const int py[2] = {Y0i + (lane >> 3), Y0i + 4 + (lane >> 3)};
  const float Xc = (float)X0i + 7.5f, Yc = (float)Y0i + 3.5f;  // centre of the strip: origin of the records
  const RnLane L = rn_lane(lane);

  float2 T[2], Cr[2], Cg[2], Cb[2];  // [c], packed over r
  // [k]: entries consumed = the whole list unless a stop says less.  A pixel is still running at list position pos
  // iff pos <= last[k]; pixels outside the image never run (0).
  uint32_t last[4];
#pragma unroll
  for (int c = 0; c < 2; c++) {
    T[c] = make_float2(1.f, 1.f);
    Cr[c] = Cg[c] = Cb[c] = make_float2(0.f, 0.f);
  }
#pragma unroll
  for (int k = 0; k < 4; k++) last[k] = (px[k & 1] < W && py[k >> 1] < H) ? (uint32_t)n : 0u;
  uint32_t live_sb = 0;  // warp-uniform: bit k set = sub-block k has a running pixel
#pragma unroll
  for (int k = 0; k < 4; k++)
    if (__any_sync(0xffffffffu, last[k] != 0u)) live_sb |= 1u << k;

  if (n > 0 && live_sb) {
    // prologue: gather of batch 0 in flight, ids of batch 1 in a register
    if (lane < n) rn_stage_issue(stage, lane, ids[lane], means2d, conic_opacity, rgb, masks);
    rn_cp_async_commit();
    uint32_t id_nxt = 32 + lane < n ? ids[32 + lane] : 0u;

    for (int base = 0; base < n; base += 32) {
      rn_cp_async_wait_all();  // this lane's entry of the current batch has landed
      __syncwarp();            // every lane is done reading the previous batch's records
      uint32_t m4 = 0;
      if (base + lane < n) {
        const RnRaw raw = rn_stage_read(stage, lane);
        // an entry with M = 0 changes neither C nor T and cannot stop a pixel: dropped here
        if (raw.m != 0.f) {
          RnRecord rec = rn_make_record(raw, Xc, Yc);
          m4 = rn_subblock_mask(rec) & live_sb;
          rec.d.x = __uint_as_float(m4);
          if (m4) buf[lane] = rec;
        }
      }
      // gather of the next batch and id load of the one after, in flight during the blend loop
      if (base + 32 + lane < n) rn_stage_issue(stage, lane, id_nxt, means2d, conic_opacity, rgb, masks);
      rn_cp_async_commit();
      id_nxt = base + 64 + lane < n ? ids[base + 64 + lane] : 0u;
      __syncwarp();  // records visible to the whole warp
      uint32_t todo = __ballot_sync(0xffffffffu, m4 != 0);
      while (todo) {
        const int jj = __ffs(todo) - 1;
        todo &= todo - 1;
        const float4 ra = buf[jj].a, rb = buf[jj].b, rc = buf[jj].c;
        // the same record is read by every lane: a warp reduction hands the compiler that fact (uniform branches)
        const uint32_t sb = __reduce_or_sync(0xffffffffu, __float_as_uint(buf[jj].d.x)) & live_sb;
        const float hi = rb.z, cap = rb.w, m = rc.w;
        const uint32_t pos = (uint32_t)(base + jj + 1);
        const RnPartial p = rn_partial(ra, rb, L);
#pragma unroll
        for (int c = 0; c < 2; c++) {
          if (sb & (5u << c)) {  // sub-block c or c + 2 reachable and live
            const float2 e = rn_eval_pair(p, L, c);
            const bool pass0 = rn_filter(e.x, hi) && pos <= last[c];
            const bool pass1 = rn_filter(e.y, hi) && pos <= last[c + 2];
            if (__any_sync(0xffffffffu, pass0 | pass1)) {
              // branch-free inside the section: a pixel that fails the filter blends with alpha = 0 (w = 0, T' = T)
              float2 alpha;
              alpha.x = pass0 ? fminf(cap, rn_ex2(e.x)) : 0.f;
              alpha.y = pass1 ? fminf(cap, rn_ex2(e.y)) : 0.f;
              const float2 a = rn_mul2(rn_splat(m), alpha);
              const float2 Tn = rn_fma2(make_float2(-a.x, -a.y), T[c], T[c]);  // T (1 - a)
              const bool stop0 = pass0 && Tn.x < MG_T_MIN, stop1 = pass1 && Tn.y < MG_T_MIN;
              float2 w = rn_mul2(a, T[c]);  // this entry is not blended if it stops the pixel; pos - 1 entries were consumed
              w.x = stop0 ? 0.f : w.x;
              w.y = stop1 ? 0.f : w.y;
              Cr[c] = rn_fma2(w, rn_splat(rc.x), Cr[c]);
              Cg[c] = rn_fma2(w, rn_splat(rc.y), Cg[c]);
              Cb[c] = rn_fma2(w, rn_splat(rc.z), Cb[c]);
              T[c].x = stop0 ? T[c].x : Tn.x;
              T[c].y = stop1 ? T[c].y : Tn.y;
              last[c] = stop0 ? pos - 1 : last[c];
              last[c + 2] = stop1 ? pos - 1 : last[c + 2];
            }
          }
        }
      }
      // refresh the live sub-blocks once per batch
      live_sb = 0;
#pragma unroll
      for (int k = 0; k < 4; k++)
        if (__any_sync(0xffffffffu, last[k] == (uint32_t)n)) live_sb |= 1u << k;
      if (!live_sb) break;
    }
    rn_cp_async_wait_all();
  }

  const size_t plane = (size_t)W * H;
#pragma unroll
  for (int k = 0; k < 4; k++) {
    const int x = px[k & 1], y = py[k >> 1];
    if (x < W && y < H) {  // (n_contrib of a pixel of an empty list: last = n = 0)
      const size_t pix = (size_t)y * W + x;
      const int c = k & 1;
      const float Tk = (k >> 1) ? T[c].y : T[c].x;
      image[pix] = fmaf(Tk, bg0, (k >> 1) ? Cr[c].y : Cr[c].x);
      image[plane + pix] = fmaf(Tk, bg1, (k >> 1) ? Cg[c].y : Cg[c].x);
      image[2 * plane + pix] = fmaf(Tk, bg2, (k >> 1) ? Cb[c].y : Cb[c].x);
      final_T[pix] = Tk;
      n_contrib[pix] = last[k];
    }
  }
}

}  // namespace

extern "C" int mg_render_fwd(const mg_camera* cam, const uint32_t* sorted_ids, const uint32_t* tile_ranges,
                             const uint32_t* tile_order, const float* means2d, const float* conic_opacity, const float* rgb, const float* masks,
                             float* image, float* final_T, uint32_t* n_contrib, void* stream) {
  if (int rc = mg_check_camera(cam)) return rc;
  MG_REQUIRE(tile_ranges && image && final_T && n_contrib, "null output or tile_ranges");
  // splat arrays are dereferenced only through non-empty tile ranges (they may be null when N = 0)
  const int gw = mg_grid_w(cam), gh = mg_grid_h(cam);
  render_fwd_kernel<<<gw * gh, RN_THREADS, 0, (cudaStream_t)stream>>>(
      cam->width, cam->height, gw, cam->bg[0], cam->bg[1], cam->bg[2], sorted_ids, (const uint2*)tile_ranges,
      tile_order, (const float2*)means2d, (const float4*)conic_opacity, rgb, masks, image, final_T, n_contrib);
  MG_CHECK_LAUNCH();
  return MG_OK;
}
