// preprocess.cu -- mg_preprocess: activate + EWA-project + SH colour + 3-sigma tile bounds.
// Steps a1-a3 of the hot path (PAPER.md:64-66 sec. 3.1, :74; O1-O8).  HBM-bound: one thread per
// Gaussian.  Geometry first (44 B); then the 192-byte SH rows of the VISIBLE Gaussians only, read with
// coalesced 128-bit loads through shared memory (a culled Gaussian never touches its row).
#include "mg_common.cuh"

namespace {

template <int D>
__device__ __forceinline__ void sh_basis(float x, float y, float z, float* Y) {
  Y[0] = MG_SH_C0;
  if (D >= 1) {
    Y[1] = -MG_SH_C1 * y;
    Y[2] = MG_SH_C1 * z;
    Y[3] = -MG_SH_C1 * x;
  }
  if (D >= 2) {
    const float xx = x * x, yy = y * y, zz = z * z;
    Y[4] = MG_SH_C2_0 * (x * y);
    Y[5] = MG_SH_C2_1 * (y * z);
    Y[6] = MG_SH_C2_2 * (2.f * zz - xx - yy);
    Y[7] = MG_SH_C2_3 * (x * z);
    Y[8] = MG_SH_C2_4 * (xx - yy);
    if (D >= 3) {
      Y[9] = MG_SH_C3_0 * (y * (3.f * xx - yy));
      Y[10] = MG_SH_C3_1 * (x * y * z);
      Y[11] = MG_SH_C3_2 * (y * (4.f * zz - xx - yy));
      Y[12] = MG_SH_C3_3 * (z * (2.f * zz - 3.f * xx - 3.f * yy));
      Y[13] = MG_SH_C3_4 * (x * (4.f * zz - xx - yy));
      Y[14] = MG_SH_C3_5 * (z * (xx - yy));
      Y[15] = MG_SH_C3_6 * (x * (xx - 3.f * yy));
    }
  }
}

// Floats per SH row, and the row stride in shared memory (128-bit accesses of 8 consecutive lanes cover all
// banks when stride / 4 is odd; scalar accesses when the stride is odd).
template <int D>
struct ShRowLayout {
  static constexpr int K = (D + 1) * (D + 1);
  static constexpr int RK = 3 * K;
  static constexpr bool VEC = (RK % 4) == 0;  // D = 1, 3
  static constexpr int STRIDE = VEC ? (((RK / 4) % 2) ? RK : RK + 4) : ((RK % 2) ? RK : RK + 1);
};

constexpr int PP_THREADS = 128;

template <int D>
__global__ void __launch_bounds__(PP_THREADS) preprocess_kernel(
    mg_camera cam, int64_t N, const float* __restrict__ means, const float* __restrict__ log_scales,
    const float* __restrict__ quats, const float* __restrict__ opacity_logits, const float* __restrict__ sh,
    float2* __restrict__ means2d, float* __restrict__ depths, float4* __restrict__ conic_opacity,
    float* __restrict__ rgb, int32_t* __restrict__ radii, int4* __restrict__ rects,
    uint32_t* __restrict__ tiles_touched, uint8_t* __restrict__ clamped, unsigned long long* __restrict__ num_rendered) {
  typedef ShRowLayout<D> L;
  constexpr int K = L::K, RK = L::RK, STRIDE = L::STRIDE;
  __shared__ __align__(16) float rows_all[PP_THREADS / 32][32 * STRIDE];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  float* wrow = rows_all[warp];
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int64_t g0 = i - lane;  // first Gaussian of this warp
  const int nrows = (int)max((int64_t)0, min((int64_t)32, N - g0));
  uint32_t touched = 0;
  // results of the geometry phase, stored after the colour phase
  float2 m2 = make_float2(0.f, 0.f);
  float4 co = make_float4(0.f, 0.f, 0.f, 0.f);
  float col[3] = {0.f, 0.f, 0.f};
  int radius = 0;
  int4 rect = make_int4(0, 0, 0, 0);
  uint32_t clampbits = 0;
  float tz = 0.f, dirx = 0.f, diry = 0.f, dirz = 0.f;
  if (i < N) {
    const float px = means[3 * i], py = means[3 * i + 1], pz = means[3 * i + 2];
    const float4 q = __ldg(reinterpret_cast<const float4*>(quats) + i);
    const float ls0 = log_scales[3 * i], ls1 = log_scales[3 * i + 1], ls2 = log_scales[3 * i + 2];
    const float logit = opacity_logits[i];
    const float* R = cam.R;


    // O2 camera space
    const float tx = R[0] * px + R[1] * py + R[2] * pz + cam.t[0];
    const float ty = R[3] * px + R[4] * py + R[5] * pz + cam.t[1];
    tz = R[6] * px + R[7] * py + R[8] * pz + cam.t[2];
    if (tz > MG_ZNEAR) {
      // O1 activations, O3 Sigma = M M^T with M = Rot diag(s)
      const float s0 = expf(ls0), s1 = expf(ls1), s2 = expf(ls2);
      const float qinv = rsqrtf(q.x * q.x + q.y * q.y + q.z * q.z + q.w * q.w);
      const float w = q.x * qinv, x = q.y * qinv, y = q.z * qinv, z = q.w * qinv;
      const float M00 = (1.f - 2.f * (y * y + z * z)) * s0, M01 = 2.f * (x * y - w * z) * s1, M02 = 2.f * (x * z + w * y) * s2;
      const float M10 = 2.f * (x * y + w * z) * s0, M11 = (1.f - 2.f * (x * x + z * z)) * s1, M12 = 2.f * (y * z - w * x) * s2;
      const float M20 = 2.f * (x * z - w * y) * s0, M21 = 2.f * (y * z + w * x) * s1, M22 = (1.f - 2.f * (x * x + y * y)) * s2;
      // O4: rows of T = J W, then Sigma2D = (T M)(T M)^T + 0.3 I
      const float limx = MG_JCLAMP * cam.width / (2.f * cam.fx), limy = MG_JCLAMP * cam.height / (2.f * cam.fy);
      const float iz = 1.f / tz;
      const float xz = fminf(limx, fmaxf(-limx, tx * iz)), yz = fminf(limy, fmaxf(-limy, ty * iz));
      const float J00 = cam.fx * iz, J02 = -cam.fx * xz * iz;  // x~ = xz*tz  =>  -fx x~/z^2 = -fx xz / z
      const float J11 = cam.fy * iz, J12 = -cam.fy * yz * iz;
      const float T00 = J00 * R[0] + J02 * R[6], T01 = J00 * R[1] + J02 * R[7], T02 = J00 * R[2] + J02 * R[8];
      const float T10 = J11 * R[3] + J12 * R[6], T11 = J11 * R[4] + J12 * R[7], T12 = J11 * R[5] + J12 * R[8];
      const float U00 = T00 * M00 + T01 * M10 + T02 * M20, U01 = T00 * M01 + T01 * M11 + T02 * M21, U02 = T00 * M02 + T01 * M12 + T02 * M22;
      const float U10 = T10 * M00 + T11 * M10 + T12 * M20, U11 = T10 * M01 + T11 * M11 + T12 * M21, U12 = T10 * M02 + T11 * M12 + T12 * M22;
      const float n0 = U00 * U00 + U01 * U01 + U02 * U02, n1 = U10 * U10 + U11 * U11 + U12 * U12;
      const float a = n0 + MG_DILATION;
      const float b = U00 * U10 + U01 * U11 + U02 * U12;
      const float c = n1 + MG_DILATION;
      // O5 conic.  det(U U^T + h I) = |U0 x U1|^2 + h (|U0|^2 + |U1|^2) + h^2: the same number as
      // a c - b^2 (Lagrange's identity) but a sum of non-negative terms, so fp32 keeps its relative
      // accuracy for elongated splats where a c and b^2 nearly cancel.
      const float cx = U01 * U12 - U02 * U11, cy = U02 * U10 - U00 * U12, cz = U00 * U11 - U01 * U10;
      const float det = (cx * cx + cy * cy + cz * cz) + MG_DILATION * (n0 + n1) + MG_DILATION * MG_DILATION;
      if (det > 0.f) {
        const float idet = 1.f / det;
        // O6 centre in pixel-index coordinates
        const float mx = cam.fx * tx * iz + (cam.cx - 0.5f), my = cam.fy * ty * iz + (cam.cy - 0.5f);
        // O7 radius and tile rectangle
        const float mid = 0.5f * (a + c);
        const float hd = 0.5f * (a - c);
        const float lam = mid + sqrtf(fmaxf(hd * hd + b * b, MG_EIG_FLOOR));  // mid^2 - det = ((a-c)/2)^2 + b^2
        const float rad_f = ceilf(3.f * sqrtf(lam));
        const int gw = (cam.width + MG_TILE - 1) / MG_TILE, gh = (cam.height + MG_TILE - 1) / MG_TILE;
        const float inv_tile = 1.f / MG_TILE;
        const int x0 = (int)fminf((float)gw, fmaxf(0.f, floorf((mx - rad_f) * inv_tile)));
        const int x1 = (int)fminf((float)gw, fmaxf(0.f, floorf((mx + rad_f + (MG_TILE - 1)) * inv_tile)));
        const int y0 = (int)fminf((float)gh, fmaxf(0.f, floorf((my - rad_f) * inv_tile)));
        const int y1 = (int)fminf((float)gh, fmaxf(0.f, floorf((my + rad_f + (MG_TILE - 1)) * inv_tile)));
        touched = (uint32_t)((x1 - x0) * (y1 - y0));
        if (touched > 0) {
          radius = (int)fminf(rad_f, 2147483520.f);
          rect = make_int4(x0, y0, x1, y1);
          m2 = make_float2(mx, my);
          co = make_float4(c * idet, -b * idet, a * idet, 1.f / (1.f + expf(-logit)));
          // O8 direction of the unit vector camera centre -> Gaussian centre (colour: second phase)
          const float cpx = -(R[0] * cam.t[0] + R[3] * cam.t[1] + R[6] * cam.t[2]);
          const float cpy = -(R[1] * cam.t[0] + R[4] * cam.t[1] + R[7] * cam.t[2]);
          const float cpz = -(R[2] * cam.t[0] + R[5] * cam.t[1] + R[8] * cam.t[2]);
          const float dx = px - cpx, dy = py - cpy, dz = pz - cpz;
          const float dinv = rsqrtf(dx * dx + dy * dy + dz * dz);
          dirx = dx * dinv; diry = dy * dinv; dirz = dz * dinv;
        }
      }
    }
  }
  // ---- colour phase: the SH rows of the warp's VISIBLE Gaussians, read by flat position with coalesced
  // 128-bit loads (a warp's 32 rows are contiguous), staged in shared memory, one row per lane
  const uint32_t vmask = __ballot_sync(0xffffffffu, touched > 0);
  if (nrows > 0 && vmask) {
    if constexpr (L::VEC) {
      const float4* src = reinterpret_cast<const float4*>(sh + g0 * RK);
#pragma unroll
      for (int k = 0; k < RK / 4; k++) {
        const int f = k * 32 + lane, g = f / (RK / 4), c = f % (RK / 4);
        if (g < nrows && ((vmask >> g) & 1u)) *reinterpret_cast<float4*>(wrow + g * STRIDE + 4 * c) = __ldg(src + f);
      }
    } else {
      const float* src = sh + g0 * RK;
#pragma unroll
      for (int k = 0; k < RK; k++) {
        const int f = k * 32 + lane, g = f / RK, c = f % RK;
        if (g < nrows && ((vmask >> g) & 1u)) wrow[g * STRIDE + c] = __ldg(src + f);
      }
    }
  }
  __syncwarp();
  if (touched > 0) {
    const float* myrow = wrow + lane * STRIDE;
    float shv[RK];
    if constexpr (L::VEC) {
#pragma unroll
      for (int j = 0; j < RK / 4; j++) {
        const float4 v = *reinterpret_cast<const float4*>(myrow + 4 * j);
        shv[4 * j] = v.x; shv[4 * j + 1] = v.y; shv[4 * j + 2] = v.z; shv[4 * j + 3] = v.w;
      }
    } else {
#pragma unroll
      for (int j = 0; j < RK; j++) shv[j] = myrow[j];
    }
    float Y[K];
    sh_basis<D>(dirx, diry, dirz, Y);
#pragma unroll
    for (int k = 0; k < 3; k++) {
      float v = 0.5f;
#pragma unroll
      for (int j = 0; j < K; j++) v = fmaf(Y[j], shv[3 * j + k], v);
      if (v < 0.f) { v = 0.f; clampbits |= 1u << k; }
      col[k] = v;
    }
  }
  if (i < N) {
    means2d[i] = m2;
    depths[i] = tz;
    conic_opacity[i] = co;
    rgb[3 * i] = col[0]; rgb[3 * i + 1] = col[1]; rgb[3 * i + 2] = col[2];
    radii[i] = radius;
    rects[i] = rect;
    tiles_touched[i] = touched;
    clamped[i] = (uint8_t)clampbits;
  }
  // R = sum of tiles_touched: warp reduction, then one atomic per warp into the caller's counter
  if (num_rendered) {
    unsigned long long t64 = touched;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) t64 += __shfl_xor_sync(0xffffffffu, t64, o);
    if ((threadIdx.x & 31) == 0 && t64) atomicAdd(num_rendered, t64);
  }
}

}  // namespace

extern "C" int mg_preprocess(const mg_camera* cam, int64_t N, const float* means, const float* log_scales,
                             const float* quats, const float* opacity_logits, const float* sh, float* means2d,
                             float* depths, float* conic_opacity, float* rgb, int32_t* radii, int32_t* rects,
                             uint32_t* tiles_touched, uint8_t* clamped, uint64_t* num_rendered,
                             uint64_t* num_rendered_host, void* stream) {
  if (int rc = mg_check_camera(cam)) return rc;
  MG_REQUIRE(N >= 0 && N < (int64_t)1 << 31, "N must be in [0, 2^31)");
  cudaStream_t st = (cudaStream_t)stream;
  MG_REQUIRE(num_rendered != nullptr || num_rendered_host == nullptr, "num_rendered_host needs the device counter num_rendered");
  if (num_rendered) MG_CHECK_CUDA(cudaMemsetAsync(num_rendered, 0, sizeof(uint64_t), st));
  if (N > 0) {
    MG_REQUIRE(means && log_scales && quats && opacity_logits && sh, "null input array");
    MG_REQUIRE(means2d && depths && conic_opacity && rgb && radii && rects && tiles_touched && clamped, "null output array");
    const int threads = PP_THREADS;
    const unsigned blocks = (unsigned)((N + threads - 1) / threads);
#define MG_LAUNCH(D)                                                                                              \
  preprocess_kernel<D><<<blocks, threads, 0, st>>>(*cam, N, means, log_scales, quats, opacity_logits, sh,         \
                                                   (float2*)means2d, depths, (float4*)conic_opacity, rgb, radii,  \
                                                   (int4*)rects, tiles_touched, clamped,      \
                                                   (unsigned long long*)num_rendered)
    switch (cam->sh_degree) {
      case 0: MG_LAUNCH(0); break;
      case 1: MG_LAUNCH(1); break;
      case 2: MG_LAUNCH(2); break;
      default: MG_LAUNCH(3); break;
    }
#undef MG_LAUNCH
    MG_CHECK_LAUNCH();
  }
  if (num_rendered_host)
    MG_CHECK_CUDA(cudaMemcpyAsync(num_rendered_host, num_rendered, sizeof(uint64_t), cudaMemcpyDeviceToHost, st));
  return MG_OK;
}
