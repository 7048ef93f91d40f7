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
// FP32-pipe and shuffle bound.  Same block geometry, staging and warp-level cull as the forward
// kernel (render_common.cuh).  A lane sums its 4 pixels in registers; the 10 per-entry sums are then
// reduced over the warp by a transposing butterfly (12 shuffles instead of 50) that leaves sum s in
// lane pair s, and 10 lanes issue one red.global.add each.
#include "render_common.cuh"

namespace {

struct BwdTargets {
  float* base[10];
  int stride[10];
  int offset[10];
};

// Sum each of 10 per-lane values over the 32 lanes.  Returns, in lanes whose slot (see rn_slot_of_lane)
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

__global__ void __launch_bounds__(RN_THREADS) render_bwd_kernel(
    int W, int H, int gw, float bg0, float bg1, float bg2, const uint32_t* __restrict__ sorted_ids,
    const uint2* __restrict__ tile_ranges, const float2* __restrict__ means2d,
    const float4* __restrict__ conic_opacity, const float* __restrict__ rgb, const float* __restrict__ masks,
    const float* __restrict__ final_T, const uint32_t* __restrict__ n_contrib, const float* __restrict__ dL_dimage,
    BwdTargets tg) {
  __shared__ RnRecord buf[2][RN_BATCH];
  __shared__ uint32_t ids_sh[2][RN_BATCH];
  __shared__ uint32_t wmax_sh[RN_THREADS / 32];
  const int tile = blockIdx.x;
  const int tx = tile % gw, ty = tile / gw;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint2 range = tile_ranges[tile];
  const uint32_t* ids = sorted_ids + range.x;

  const int px0 = tx * MG_TILE + 2 * (lane & 7), py0 = ty * MG_TILE + 8 * warp + 2 * (lane >> 3);
  const float fx0 = (float)px0, fx1 = (float)(px0 + 1), fy0 = (float)py0, fy1 = (float)(py0 + 1);
  const float X0 = (float)(tx * MG_TILE), Y0 = (float)(ty * MG_TILE + 8 * warp);

  // per-pixel state
  float T[4], gB[4], g0[4], g1[4], g2[4], tfg[4];
  uint32_t last[4];
  const size_t plane = (size_t)W * H;
  uint32_t lmax = 0;
#pragma unroll
  for (int k = 0; k < 4; k++) {
    const int px = px0 + (k & 1), py = py0 + (k >> 1);
    T[k] = 1.f; gB[k] = 0.f; g0[k] = g1[k] = g2[k] = 0.f; tfg[k] = 0.f; last[k] = 0;
    if (px < W && py < H) {
      const size_t pix = (size_t)py * W + px;
      T[k] = final_T[pix];
      last[k] = n_contrib[pix];
      g0[k] = dL_dimage[pix];
      g1[k] = dL_dimage[plane + pix];
      g2[k] = dL_dimage[2 * plane + pix];
      tfg[k] = T[k] * (g0[k] * bg0 + g1[k] * bg1 + g2[k] * bg2);  // T_{N+1} g.c_bg
    }
    lmax = max(lmax, last[k]);
  }
  const uint32_t wmax = __reduce_max_sync(0xffffffffu, lmax);
  if (lane == 0) wmax_sh[warp] = wmax;
  __syncthreads();
  uint32_t bmax = 0;
#pragma unroll
  for (int w = 0; w < RN_THREADS / 32; w++) bmax = max(bmax, wmax_sh[w]);
  bmax = min(bmax, range.y - range.x);  // never walk past the tile's own list
  if (bmax == 0) return;

  // where this lane's reduced sum goes
  const int slot = slot_of_lane(lane);
  float* tgt_base = nullptr;
  int tgt_stride = 0, tgt_off = 0;
#pragma unroll
  for (int s = 0; s < 10; s++)
    if (slot == s) { tgt_base = tg.base[s]; tgt_stride = tg.stride[s]; tgt_off = tg.offset[s]; }

  const int n = (int)bmax;  // entries at positions > bmax are never visited
  const int bstart = (n - 1) / RN_BATCH;
  uint32_t id_next[2];
#pragma unroll
  for (int s = 0; s < 2; s++) {
    const int k = s * RN_THREADS + threadIdx.x;
    const int i0 = bstart * RN_BATCH + k;
    if (i0 < n) {
      const uint32_t id = ids[i0];
      ids_sh[0][k] = id;
      buf[0][k] = rn_make_record(rn_gather(id, means2d, conic_opacity, rgb, masks));
    }
    const int i1 = (bstart - 1) * RN_BATCH + k;
    id_next[s] = bstart >= 1 ? ids[i1] : 0u;
  }
  __syncthreads();

  int cur = 0;
  for (int b = bstart; b >= 0; b--) {
    const int base = b * RN_BATCH;
    const int cnt = min(RN_BATCH, n - base);
    RnRaw raw[2];
    uint32_t id_next2[2];
#pragma unroll
    for (int s = 0; s < 2; s++) {
      const int k = s * RN_THREADS + threadIdx.x;
      if (b >= 1) raw[s] = rn_gather(id_next[s], means2d, conic_opacity, rgb, masks);
      id_next2[s] = b >= 2 ? ids[(b - 2) * RN_BATCH + k] : 0u;
    }

    const RnRecord* rec = buf[cur];
    for (int c0 = ((cnt - 1) >> 5) << 5; c0 >= 0; c0 -= 32) {
      const int j = c0 + lane;
      bool keep = false;
      if (j < cnt && (uint32_t)(base + j + 1) <= wmax) {
        const float4 ra = rec[j].a, rb = rec[j].b;
        keep = rn_max_e_over_strip(ra, rb, X0, Y0) >= RN_LOG2_ALPHA_MIN - RN_CULL_SLACK;
      }
      uint32_t todo = __ballot_sync(0xffffffffu, keep);
      while (todo) {
        const int bit = 31 - __clz(todo);
        todo &= ~(1u << bit);
        const int jj = c0 + bit;
        const float4 ra = rec[jj].a, rb = rec[jj].b;
        const float lo = rb.y;
        float dx[2], dy[2], e[4];
        rn_eval_quad(ra, rb, fx0, fx1, fy0, fy1, dx, dy, e);
        uint32_t pass = rn_filter_quad(e, lo);
        const uint32_t pos = (uint32_t)(base + jj + 1);
#pragma unroll
        for (int k = 0; k < 4; k++)
          if (pos > last[k]) pass &= ~(1u << k);
        if (!__any_sync(0xffffffffu, pass != 0)) continue;

        const float4 rc = rec[jj].c;
        const float m = rb.z;
        float S = 0.f, Sx = 0.f, Sy = 0.f, Sxx = 0.f, Sxy = 0.f, Syy = 0.f;
        float dr = 0.f, dg = 0.f, db = 0.f, dm = 0.f;
#pragma unroll
        for (int k = 0; k < 4; k++) {
          if (pass >> k & 1u) {
            const float raw_alpha = rn_ex2(e[k]);
            const float alpha = fminf(MG_ALPHA_MAX, raw_alpha);
            const float a = m * alpha;
            const float oma = 1.f - a;
            const float inv = __frcp_rn(oma);
            const float Ti = T[k] * inv;
            const float gc = g0[k] * rc.x + g1[k] * rc.y + g2[k] * rc.z;
            const float X = Ti * (gc - gB[k]) - tfg[k] * inv;
            dm = fmaf(alpha, X, dm);
            const float wgt = a * Ti;
            dr = fmaf(wgt, g0[k], dr);
            dg = fmaf(wgt, g1[k], dg);
            db = fmaf(wgt, g2[k], db);
            gB[k] = fmaf(a, gc, oma * gB[k]);
            T[k] = Ti;
            if (raw_alpha <= MG_ALPHA_MAX) {
              const float q = alpha * (m * X);
              const float ddx = dx[k & 1], ddy = dy[k >> 1];
              const float qx = q * ddx, qy = q * ddy;
              S += q; Sx += qx; Sy += qy;
              Sxx = fmaf(qx, ddx, Sxx);
              Sxy = fmaf(qx, ddy, Sxy);
              Syy = fmaf(qy, ddy, Syy);
            }
          }
        }
        // per-entry linear map: true conic (A,B,C) = (-2 ln2 A2, -ln2 B2, -2 ln2 C2)
        float v[10];
        v[0] = RN_LN2 * (2.f * ra.z * Sx + ra.w * Sy);   // dL/dmean2d.x = -(A Sx + B Sy)
        v[1] = RN_LN2 * (ra.w * Sx + 2.f * rb.x * Sy);   // dL/dmean2d.y = -(B Sx + C Sy)
        v[2] = -0.5f * Sxx;                              // dL/dA
        v[3] = -Sxy;                                     // dL/dB
        v[4] = -0.5f * Syy;                              // dL/dC
        v[5] = S * rb.w;                                 // dL/do = sum q / o
        v[6] = dr; v[7] = dg; v[8] = db;
        v[9] = dm;
        const float total = transpose_reduce10(v, lane);
        if (slot >= 0 && total != 0.f) {
          const uint32_t id = ids_sh[cur][jj];
          atomicAdd(tgt_base + (size_t)id * tgt_stride + tgt_off, total);
        }
      }
    }

#pragma unroll
    for (int s = 0; s < 2; s++) {
      const int k = s * RN_THREADS + threadIdx.x;
      if (b >= 1) {
        ids_sh[cur ^ 1][k] = id_next[s];
        buf[cur ^ 1][k] = rn_make_record(raw[s]);
      }
      id_next[s] = id_next2[s];
    }
    cur ^= 1;
    __syncthreads();
  }
}

}  // namespace

extern "C" int mg_render_bwd(const mg_camera* cam, int64_t N, const uint32_t* sorted_ids, const uint32_t* tile_ranges,
                             const float* means2d, const float* conic_opacity, const float* rgb, const float* masks,
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
  render_bwd_kernel<<<gw * gh, RN_THREADS, 0, st>>>(cam->width, cam->height, gw, cam->bg[0], cam->bg[1], cam->bg[2],
                                                    sorted_ids, (const uint2*)tile_ranges, (const float2*)means2d,
                                                    (const float4*)conic_opacity, rgb, masks, final_T, n_contrib,
                                                    dL_dimage, tg);
  MG_CHECK_LAUNCH();
  return MG_OK;
}
