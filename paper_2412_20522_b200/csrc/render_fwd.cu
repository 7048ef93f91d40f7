// render_fwd.cu -- mg_render_fwd: masked front-to-back blend of a 16x16 tile (step a7).
// Eq. 3-4: C += M_i alpha_i T_i c_i,  T_{i+1} = (1 - M_i alpha_i) T_i;
// Eq. 9-10: image = C + T_{N+1} c_bg.  Thresholds: DESIGN.md readings 1-5.
//
// FP32-pipe bound (no dense contraction on this path, so no tensor cores).  Design:
//  * 2 warps per tile, a 2x2 pixel quad per lane (render_common.cuh);
//  * list entries gathered one batch ahead into registers, converted to log2-domain records and
//    staged in double-buffered shared memory: one barrier per batch of 128 entries;
//  * per warp, 32 entries at a time are tested against the warp's 16x8 strip (exact maximum of the
//    concave exponent over the strip) and only the survivors are evaluated per pixel;
//  * the alpha filter is two compares on the exponent, the exponential is taken only for pairs
//    that pass; a warp leaves the loop when all its pixels have stopped.
#include "render_common.cuh"

namespace {

__global__ void __launch_bounds__(RN_THREADS) render_fwd_kernel(
    int W, int H, int gw, float bg0, float bg1, float bg2, const uint32_t* __restrict__ sorted_ids,
    const uint2* __restrict__ tile_ranges, const float2* __restrict__ means2d,
    const float4* __restrict__ conic_opacity, const float* __restrict__ rgb, const float* __restrict__ masks,
    float* __restrict__ image, float* __restrict__ final_T, uint32_t* __restrict__ n_contrib) {
  __shared__ RnRecord buf[2][RN_BATCH];
  const int tile = blockIdx.x;
  const int tx = tile % gw, ty = tile / gw;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint2 range = tile_ranges[tile];
  const int n = (int)(range.y - range.x);
  const uint32_t* ids = sorted_ids + range.x;

  // quad of this lane
  const int px0 = tx * MG_TILE + 2 * (lane & 7), py0 = ty * MG_TILE + 8 * warp + 2 * (lane >> 3);
  const float fx0 = (float)px0, fx1 = (float)(px0 + 1), fy0 = (float)py0, fy1 = (float)(py0 + 1);
  const float X0 = (float)(tx * MG_TILE), Y0 = (float)(ty * MG_TILE + 8 * warp);

  float T[4] = {1.f, 1.f, 1.f, 1.f};
  float Cr[4] = {0.f, 0.f, 0.f, 0.f}, Cg[4] = {0.f, 0.f, 0.f, 0.f}, Cb[4] = {0.f, 0.f, 0.f, 0.f};
  uint32_t last[4] = {0u, 0u, 0u, 0u};
  // bit k set = pixel k still running (k = 2*row + col).  Pixels outside the image never run.
  uint32_t live = 0;
  if (px0 < W && py0 < H) live |= 1u;
  if (px0 + 1 < W && py0 < H) live |= 2u;
  if (px0 < W && py0 + 1 < H) live |= 4u;
  if (px0 + 1 < W && py0 + 1 < H) live |= 8u;
  bool warp_done = !__any_sync(0xffffffffu, live != 0);

  const int nbatches = (n + RN_BATCH - 1) / RN_BATCH;
  // prologue: batch 0 -> buf[0]; ids of batch 1 -> registers
  uint32_t id_next[2];
#pragma unroll
  for (int s = 0; s < 2; s++) {
    const int k = s * RN_THREADS + threadIdx.x;
    if (k < n) buf[0][k] = rn_make_record(rn_gather(ids[k], means2d, conic_opacity, rgb, masks));
    const int k1 = RN_BATCH + k;
    id_next[s] = k1 < n ? ids[k1] : 0u;
  }
  __syncthreads();

  int cur = 0;
  for (int b = 0; b < nbatches; b++) {
    const int base = b * RN_BATCH;
    const int cnt = min(RN_BATCH, n - base);
    // issue the gathers of batch b+1 and the id loads of batch b+2 before computing on batch b
    RnRaw raw[2];
    uint32_t id_next2[2];
#pragma unroll
    for (int s = 0; s < 2; s++) {
      const int k = s * RN_THREADS + threadIdx.x;
      if (base + RN_BATCH + k < n) raw[s] = rn_gather(id_next[s], means2d, conic_opacity, rgb, masks);
      const int k2 = base + 2 * RN_BATCH + k;
      id_next2[s] = k2 < n ? ids[k2] : 0u;
    }

    if (!warp_done) {
      const RnRecord* rec = buf[cur];
      for (int c0 = 0; c0 < cnt; c0 += 32) {
        // warp-level cull of 32 entries against this warp's strip
        const int j = c0 + lane;
        bool keep = false;
        if (j < cnt) {
          const float4 ra = rec[j].a, rb = rec[j].b;
          keep = rn_max_e_over_strip(ra, rb, X0, Y0) >= RN_LOG2_ALPHA_MIN - RN_CULL_SLACK;
        }
        uint32_t todo = __ballot_sync(0xffffffffu, keep);
        while (todo) {
          const int jj = c0 + __ffs(todo) - 1;
          todo &= todo - 1;
          const float4 ra = rec[jj].a, rb = rec[jj].b;
          const float lo = rb.y;
          float dx[2], dy[2], e[4];
          rn_eval_quad(ra, rb, fx0, fx1, fy0, fy1, dx, dy, e);
          uint32_t pass = rn_filter_quad(e, lo);
          pass &= live;
          if (__any_sync(0xffffffffu, pass != 0)) {
            const float4 rc = rec[jj].c;
            const uint32_t pos = (uint32_t)(base + jj + 1);
#pragma unroll
            for (int k = 0; k < 4; k++) {
              if (pass >> k & 1u) {
                const float alpha = fminf(MG_ALPHA_MAX, rn_ex2(e[k]));
                const float a = rb.z * alpha;
                const float Tn = T[k] * (1.f - a);
                if (Tn < MG_T_MIN) {
                  live &= ~(1u << k);  // stop: this entry is neither blended nor counted
                } else {
                  const float w = a * T[k];
                  Cr[k] = fmaf(w, rc.x, Cr[k]);
                  Cg[k] = fmaf(w, rc.y, Cg[k]);
                  Cb[k] = fmaf(w, rc.z, Cb[k]);
                  T[k] = Tn;
                  last[k] = pos;
                }
              }
            }
          }
        }
        if (!__any_sync(0xffffffffu, live != 0)) { warp_done = true; break; }
      }
    }

    // publish batch b+1 into the other buffer
#pragma unroll
    for (int s = 0; s < 2; s++) {
      const int k = s * RN_THREADS + threadIdx.x;
      if (base + RN_BATCH + k < n) buf[cur ^ 1][k] = rn_make_record(raw[s]);
      id_next[s] = id_next2[s];
    }
    cur ^= 1;
    if (__syncthreads_and(warp_done)) break;
  }

  const size_t plane = (size_t)W * H;
#pragma unroll
  for (int k = 0; k < 4; k++) {
    const int px = px0 + (k & 1), py = py0 + (k >> 1);
    if (px < W && py < H) {
      const size_t pix = (size_t)py * W + px;
      image[pix] = fmaf(T[k], bg0, Cr[k]);
      image[plane + pix] = fmaf(T[k], bg1, Cg[k]);
      image[2 * plane + pix] = fmaf(T[k], bg2, Cb[k]);
      final_T[pix] = T[k];
      n_contrib[pix] = last[k];
    }
  }
}

}  // namespace

extern "C" int mg_render_fwd(const mg_camera* cam, const uint32_t* sorted_ids, const uint32_t* tile_ranges,
                             const float* means2d, const float* conic_opacity, const float* rgb, const float* masks,
                             float* image, float* final_T, uint32_t* n_contrib, void* stream) {
  if (int rc = mg_check_camera(cam)) return rc;
  MG_REQUIRE(tile_ranges && image && final_T && n_contrib, "null output or tile_ranges");
  // splat arrays are dereferenced only through non-empty tile ranges (they may be null when N = 0)
  const int gw = mg_grid_w(cam), gh = mg_grid_h(cam);
  render_fwd_kernel<<<gw * gh, RN_THREADS, 0, (cudaStream_t)stream>>>(
      cam->width, cam->height, gw, cam->bg[0], cam->bg[1], cam->bg[2], sorted_ids, (const uint2*)tile_ranges,
      (const float2*)means2d, (const float4*)conic_opacity, rgb, masks, image, final_T, n_contrib);
  MG_CHECK_LAUNCH();
  return MG_OK;
}
