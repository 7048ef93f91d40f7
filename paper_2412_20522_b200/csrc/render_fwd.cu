// render_fwd.cu -- mg_render_fwd: masked front-to-back blend of a 16x16 tile (step a7).
// Eq. 3-4: C += M_i alpha_i T_i c_i,  T_{i+1} = (1 - M_i alpha_i) T_i;
// Eq. 9-10: image = C + T_{N+1} c_bg.  Thresholds: DESIGN.md readings 1-5.
//
// FP32-issue bound (no dense contraction on this path, so no tensor cores).  Design (render_common.cuh):
//  * 2 independent warps per tile, each a 16x8 strip of four 8x4 sub-blocks, one pixel of each per lane;
//  * an entry with M = 0 changes neither C nor T and cannot stop a pixel, and n_contrib counts the
//    entries consumed before the stop (include/mg.h, reading 5), so the forward pass owes masked entries nothing.  They
//    are removed BEFORE anything expensive happens: the warp classifies its list 64 entries at a time -- ids from a
//    register prefetch, only the 4-byte mask of each entry gathered (cp.async) -- and a ballot appends the survivors'
//    (id, list position, M) to a small ring queue in shared memory;
//  * the attributes are gathered (cp.async, one batch ahead) for full batches of 32 UNMASKED entries taken from the
//    queue; each lane expands its entry's record about the strip's centre and computes its 4-bit sub-block reach mask
//    (lanes = entries), a ballot, then the surviving entries are walked in list order;
//  * per surviving entry only the reachable, still-live pairs of sub-blocks are evaluated, two pixels per packed
//    FP32 instruction; the alpha filter is two compares on the exponent, the exponential is taken only for pixels
//    that pass;
//  * a warp leaves when all its pixels have stopped.
#include "render_common.cuh"

#ifndef RN_FWD_MINB
#define RN_FWD_MINB 12  // minimum resident blocks per SM asked of ptxas (register budget): 72 registers, 14 blocks resident.
                        // Measured: 10 -> 80 registers, 12 blocks: equal; 16 -> 64 registers, 16 blocks: 10 % SLOWER
                        // (shared memory grows with the blocks and comes out of the L1 the gathers live on)
#endif

namespace {

// Per-warp ring queue of the list's unmasked entries that have not been turned into records yet, and the landing
// zone of one classification step.  A step never finds more than 31 entries waiting (a full batch would have been
// taken first) and adds at most FQ_STEP, so FQ_CAP = 128 slots are never overrun.
constexpr int FQ_STEP = 64;
constexpr int FQ_CAP = 128;
struct FwdQueue {
  uint32_t id[FQ_CAP];
  uint32_t pos[FQ_CAP];  // 1-based position in the tile's list
  float m[FQ_CAP];
  uint32_t rid[FQ_STEP];  // ids of the step whose masks are in flight
  float land[FQ_STEP];    // its masks (cp.async)
};

__device__ __forceinline__ RnRaw rn_stage_read_attr(const RnStage* s, int lane) {
  RnRaw v;
  v.m2 = s->m2[lane];
  v.co = s->co[lane];
  v.r = s->rgb[lane][0];
  v.g = s->rgb[lane][1];
  v.b = s->rgb[lane][2];
  v.m = 0.f;
  return v;
}

__global__ void __launch_bounds__(RN_THREADS, RN_FWD_MINB) render_fwd_kernel(
    int W, int H, int gw, float bg0, float bg1, float bg2, const uint32_t* __restrict__ sorted_ids,
    const uint2* __restrict__ tile_ranges, const uint32_t* __restrict__ tile_order,
    const float2* __restrict__ means2d, const float4* __restrict__ conic_opacity, const float* __restrict__ rgb,
    const float* __restrict__ masks, float* __restrict__ image, float* __restrict__ final_T, uint32_t* __restrict__ n_contrib) {
  __shared__ RnRecord buf_all[RN_WARPS][32];
  __shared__ RnStage stage_all[RN_WARPS];
  __shared__ FwdQueue queue_all[RN_WARPS];
  const int tile = tile_order ? (int)tile_order[blockIdx.x] : (int)blockIdx.x;  // longest lists first
  const int tx = tile % gw, ty = tile / gw;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  RnRecord* buf = buf_all[warp];
  RnStage* stage = &stage_all[warp];
  FwdQueue* Q = &queue_all[warp];
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
    // ---- classification of the list, FQ_STEP entries per step (two per lane)
    int rnext = 0;         // first list position (0-based) of the next step to be issued
    int rland = -1;        // first list position of the step whose masks are in flight / have landed (-1: none)
    int qhead = 0, qcount = 0;  // ring queue of unmasked entries not yet turned into records
    uint32_t idA = lane < n ? ids[lane] : 0u, idB = 32 + lane < n ? ids[32 + lane] : 0u;  // ids of step rnext
    // the masks of a step are gathered into Q->land; its ids are kept beside them until the step is classified
    auto issue_step = [&]() {
      Q->rid[lane] = idA;
      Q->rid[32 + lane] = idB;
      if (rnext + lane < n) rn_cp_async(&Q->land[lane], masks + idA, 4);
      if (rnext + 32 + lane < n) rn_cp_async(&Q->land[32 + lane], masks + idB, 4);
      rland = rnext;
      rnext += FQ_STEP;
      idA = rnext + lane < n ? ids[rnext + lane] : 0u;  // ids of the step after, in flight until that step is issued
      idB = rnext + 32 + lane < n ? ids[rnext + 32 + lane] : 0u;
    };
    auto classify_step = [&]() {  // the step at rland has landed
      const int p0 = rland + lane, p1 = rland + 32 + lane;
      const float m0 = p0 < n ? Q->land[lane] : 0.f, m1 = p1 < n ? Q->land[32 + lane] : 0.f;
      const uint32_t b0 = __ballot_sync(0xffffffffu, m0 != 0.f), b1 = __ballot_sync(0xffffffffu, m1 != 0.f);
      const uint32_t lt = (1u << lane) - 1u;
      const int tail = qhead + qcount;
      if (m0 != 0.f) {
        const int s = (tail + __popc(b0 & lt)) & (FQ_CAP - 1);
        Q->id[s] = Q->rid[lane]; Q->pos[s] = (uint32_t)(p0 + 1); Q->m[s] = m0;
      }
      if (m1 != 0.f) {
        const int s = (tail + __popc(b0) + __popc(b1 & lt)) & (FQ_CAP - 1);
        Q->id[s] = Q->rid[32 + lane]; Q->pos[s] = (uint32_t)(p1 + 1); Q->m[s] = m1;
      }
      qcount += __popc(b0) + __popc(b1);
      rland = -1;
      __syncwarp();  // queue entries visible to the lanes that will gather them; land / rid free for the next step
    };
    // Fills the queue to a full batch (or to the end of the list), issues the attribute gather of the next batch (its
    // size is returned) and keeps the mask gather of one step in flight.  Only the first step classified here can
    // have been in flight already; a further one costs a round trip, which other warps cover.  Invariant: at most ONE
    // step is issued and not yet classified (rland >= 0), because rid / land hold exactly one step.
    auto refill_and_issue = [&]() -> int {
      while (qcount < 32 && (rland >= 0 || rnext < n)) {
        if (rland < 0) issue_step();
        rn_cp_async_commit();
        rn_cp_async_wait_all();
        __syncwarp();
        classify_step();
      }
      const int nb = min(32, qcount);
      if (lane < nb) rn_stage_issue_attr(stage, lane, Q->id[(qhead + lane) & (FQ_CAP - 1)], means2d, conic_opacity, rgb);
      // one more step of masks in flight -- unless one is still waiting to be classified (the queue was full enough
      // without it): its ids and landing zone must not be overwritten
      if (rland < 0 && rnext < n) issue_step();
      rn_cp_async_commit();
      return nb;
    };

    int nb = refill_and_issue();  // prologue: batch 0 in flight
    while (nb > 0) {
      rn_cp_async_wait_all();  // this lane's entry of the current batch has landed (and the masks of the step in flight)
      __syncwarp();            // every lane is done reading the previous batch's records
      uint32_t m4 = 0;
      if (lane < nb) {
        const int s = (qhead + lane) & (FQ_CAP - 1);
        RnRaw raw = rn_stage_read_attr(stage, lane);
        raw.m = Q->m[s];
        RnRecord rec = rn_make_record(raw, Xc, Yc);
        m4 = rn_subblock_mask(rec) & live_sb;
        rec.d.x = __uint_as_float(m4);
        rec.d.w = __uint_as_float(Q->pos[s]);  // 1-based list position (the record's 1/o slot: unused by the forward pass)
        if (m4) buf[lane] = rec;
      }
      qhead = (qhead + nb) & (FQ_CAP - 1);
      qcount -= nb;
      __syncwarp();  // this batch's queue slots have been read by every lane before classification reuses any
      // next batch: queue refill, attribute gather, one more step of masks -- all in flight during the blend loop
      nb = refill_and_issue();
      __syncwarp();  // records visible to the whole warp
      uint32_t todo = __ballot_sync(0xffffffffu, m4 != 0);
      while (todo) {
        const int jj = __ffs(todo) - 1;
        todo &= todo - 1;
        const float4 ra = buf[jj].a, rb = buf[jj].b, rc = buf[jj].c;
        // the same record is read by every lane: a warp reduction hands the compiler that fact (uniform branches)
        const uint32_t sb = __reduce_or_sync(0xffffffffu, __float_as_uint(buf[jj].d.x)) & live_sb;
        const float hi = rb.z, cap = rb.w, m = rc.w;
        const uint32_t pos = __float_as_uint(buf[jj].d.w);  // the entry's position in the tile's list
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
