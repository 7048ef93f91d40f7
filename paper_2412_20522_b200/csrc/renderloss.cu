// renderloss.cu -- mg_render_loss: L_render and dL/dimage on the device.
// Eq. 8 adds lambda_m L_m to "the original rendering loss", which the paper does not define;
// reading 26: the loss of the 3DGS method it modifies,
//     L_render = (1 - lambda) mean|I - G| + lambda (1 - mean SSIM(I, G)),
// SSIM per channel with a separable 11-tap Gaussian window (sigma 1.5), zero padding, C1 = 0.01^2, C2 = 0.03^2.
// Two kernels over 16x16 pixel tiles (+5 pixels of halo staged in shared memory), both HBM-bound:
//   forward : five filtered maps (I, G, I^2, G^2, IG) -> SSIM, sums of SSIM and |I - G|, and the three partial
//             derivative maps dSSIM/d(mu1, E[I^2], E[IG]);
//   backward: the three maps filtered again (the window is symmetric, so the adjoint is the same filter) and
//             combined with the L1 sign into dL/dI.
#include "mg_common.cuh"

namespace {

constexpr int RL_T = 16;              // tile side
constexpr int RL_R = 5;               // window radius (11 taps)
constexpr int RL_S = RL_T + 2 * RL_R; // staged side: 26
constexpr float RL_C1 = 0.01f * 0.01f, RL_C2 = 0.03f * 0.03f;

__constant__ float c_win[2 * RL_R + 1];

// Stage a (RL_S x RL_S) window of plane `src` around the tile at (x0, y0); zero outside the image.
__device__ __forceinline__ void stage(const float* __restrict__ src, int W, int H, int x0, int y0, float (*dst)[RL_S]) {
  for (int i = threadIdx.y * RL_T + threadIdx.x; i < RL_S * RL_S; i += RL_T * RL_T) {
    const int r = i / RL_S, c = i - r * RL_S;
    const int y = y0 - RL_R + r, x = x0 - RL_R + c;
    dst[r][c] = (x >= 0 && x < W && y >= 0 && y < H) ? src[(size_t)y * W + x] : 0.f;
  }
}

__global__ void __launch_bounds__(RL_T * RL_T) ssim_fwd_kernel(int W, int H, const float* __restrict__ img,
                                                               const float* __restrict__ tgt, float* __restrict__ d_mu1,
                                                               float* __restrict__ d_e1, float* __restrict__ d_e12,
                                                               double* __restrict__ stats) {
  __shared__ float sx[RL_S][RL_S], sy[RL_S][RL_S];
  __shared__ float hz[5][RL_S][RL_T];  // horizontally filtered I, G, I^2, G^2, IG
  __shared__ double red[2][RL_T * RL_T / 32];
  const size_t plane = (size_t)W * H;
  const float* px = img + blockIdx.z * plane;
  const float* py = tgt + blockIdx.z * plane;
  const int x0 = blockIdx.x * RL_T, y0 = blockIdx.y * RL_T;
  stage(px, W, H, x0, y0, sx);
  stage(py, W, H, x0, y0, sy);
  __syncthreads();
  for (int i = threadIdx.y * RL_T + threadIdx.x; i < RL_S * RL_T; i += RL_T * RL_T) {
    const int r = i / RL_T, c = i - r * RL_T;
    float a0 = 0.f, a1 = 0.f, a2 = 0.f, a3 = 0.f, a4 = 0.f;
#pragma unroll
    for (int k = 0; k <= 2 * RL_R; k++) {
      const float w = c_win[k], x = sx[r][c + k], y = sy[r][c + k];
      a0 = fmaf(w, x, a0); a1 = fmaf(w, y, a1);
      a2 = fmaf(w, x * x, a2); a3 = fmaf(w, y * y, a3); a4 = fmaf(w, x * y, a4);
    }
    hz[0][r][c] = a0; hz[1][r][c] = a1; hz[2][r][c] = a2; hz[3][r][c] = a3; hz[4][r][c] = a4;
  }
  __syncthreads();
  const int tx = threadIdx.x, ty = threadIdx.y;
  float mu1 = 0.f, mu2 = 0.f, e1 = 0.f, e2 = 0.f, e12 = 0.f;
#pragma unroll
  for (int k = 0; k <= 2 * RL_R; k++) {
    const float w = c_win[k];
    mu1 = fmaf(w, hz[0][ty + k][tx], mu1); mu2 = fmaf(w, hz[1][ty + k][tx], mu2);
    e1 = fmaf(w, hz[2][ty + k][tx], e1); e2 = fmaf(w, hz[3][ty + k][tx], e2); e12 = fmaf(w, hz[4][ty + k][tx], e12);
  }
  const int x = x0 + tx, y = y0 + ty;
  const bool in = x < W && y < H;
  double ssim_d = 0.0, l1_d = 0.0;
  if (in) {
    const float s1 = e1 - mu1 * mu1, s2 = e2 - mu2 * mu2, s12 = e12 - mu1 * mu2;
    const float A = 2.f * mu1 * mu2 + RL_C1, B = 2.f * s12 + RL_C2;
    const float C = mu1 * mu1 + mu2 * mu2 + RL_C1, D = s1 + s2 + RL_C2;
    const float iCD = 1.f / (C * D);
    const size_t p = blockIdx.z * plane + (size_t)y * W + x;
    d_mu1[p] = (2.f * mu2 * (B - A)) * iCD - A * B * iCD * iCD * (2.f * mu1 * (D - C));
    d_e1[p] = -A * B * iCD / D;
    d_e12[p] = 2.f * A * iCD;
    ssim_d = (double)(A * B * iCD);
    l1_d = (double)fabsf(sx[ty + RL_R][tx + RL_R] - sy[ty + RL_R][tx + RL_R]);
  }
#pragma unroll
  for (int o = 16; o >= 1; o >>= 1) {
    ssim_d += __shfl_xor_sync(0xffffffffu, ssim_d, o);
    l1_d += __shfl_xor_sync(0xffffffffu, l1_d, o);
  }
  const int t = ty * RL_T + tx;
  if ((t & 31) == 0) { red[0][t >> 5] = l1_d; red[1][t >> 5] = ssim_d; }
  __syncthreads();
  if (t == 0) {
    double a = 0.0, b = 0.0;
#pragma unroll
    for (int w = 0; w < RL_T * RL_T / 32; w++) { a += red[0][w]; b += red[1][w]; }
    atomicAdd(&stats[0], a);
    atomicAdd(&stats[1], b);
  }
}

// stats: [0] sum|I-G| -> mean, [1] sum SSIM -> mean, [2] = loss
__global__ void loss_finalize_kernel(double* __restrict__ stats, double n, double lambda) {
  const double l1 = stats[0] / n, ssim = stats[1] / n;
  stats[0] = l1; stats[1] = ssim;
  stats[2] = (1.0 - lambda) * l1 + lambda * (1.0 - ssim);
}

__global__ void __launch_bounds__(RL_T * RL_T) ssim_bwd_kernel(int W, int H, const float* __restrict__ img,
                                                               const float* __restrict__ tgt, const float* __restrict__ d_mu1,
                                                               const float* __restrict__ d_e1, const float* __restrict__ d_e12,
                                                               float w_l1, float w_ssim, float* __restrict__ dL_dimage) {
  __shared__ float sm[3][RL_S][RL_S];
  __shared__ float hz[3][RL_S][RL_T];
  const size_t plane = (size_t)W * H, off = blockIdx.z * plane;
  const int x0 = blockIdx.x * RL_T, y0 = blockIdx.y * RL_T;
  stage(d_mu1 + off, W, H, x0, y0, sm[0]);
  stage(d_e1 + off, W, H, x0, y0, sm[1]);
  stage(d_e12 + off, W, H, x0, y0, sm[2]);
  __syncthreads();
  for (int i = threadIdx.y * RL_T + threadIdx.x; i < RL_S * RL_T; i += RL_T * RL_T) {
    const int r = i / RL_T, c = i - r * RL_T;
    float a0 = 0.f, a1 = 0.f, a2 = 0.f;
#pragma unroll
    for (int k = 0; k <= 2 * RL_R; k++) {
      const float w = c_win[k];
      a0 = fmaf(w, sm[0][r][c + k], a0); a1 = fmaf(w, sm[1][r][c + k], a1); a2 = fmaf(w, sm[2][r][c + k], a2);
    }
    hz[0][r][c] = a0; hz[1][r][c] = a1; hz[2][r][c] = a2;
  }
  __syncthreads();
  const int tx = threadIdx.x, ty = threadIdx.y;
  float b0 = 0.f, b1 = 0.f, b2 = 0.f;
#pragma unroll
  for (int k = 0; k <= 2 * RL_R; k++) {
    const float w = c_win[k];
    b0 = fmaf(w, hz[0][ty + k][tx], b0); b1 = fmaf(w, hz[1][ty + k][tx], b1); b2 = fmaf(w, hz[2][ty + k][tx], b2);
  }
  const int x = x0 + tx, y = y0 + ty;
  if (x < W && y < H) {
    const size_t p = off + (size_t)y * W + x;
    const float xi = img[p], yi = tgt[p];
    const float d_ssim = b0 + 2.f * xi * b1 + yi * b2;
    const float sgn = xi > yi ? 1.f : (xi < yi ? -1.f : 0.f);
    dL_dimage[p] = w_l1 * sgn - w_ssim * d_ssim;
  }
}

}  // namespace

extern "C" size_t mg_render_loss_workspace_bytes(int32_t width, int32_t height) {
  if (width <= 0 || height <= 0) return 0;
  return 3 * 3 * sizeof(float) * (size_t)width * height;
}

extern "C" int mg_render_loss(int32_t width, int32_t height, const float* image, const float* target, float lambda_dssim,
                              float* dL_dimage, double* stats, void* workspace, size_t workspace_bytes, void* stream) {
  MG_REQUIRE(width > 0 && height > 0, "image size must be positive");
  MG_REQUIRE(image && target && dL_dimage && stats && workspace, "null array");
  MG_REQUIRE(lambda_dssim >= 0.f && lambda_dssim <= 1.f, "lambda_dssim must be in [0, 1]");
  if (workspace_bytes < mg_render_loss_workspace_bytes(width, height)) {
    mg_set_error("workspace too small: %zu bytes given, %zu needed", workspace_bytes, mg_render_loss_workspace_bytes(width, height));
    return MG_ERR_CAPACITY;
  }
  cudaStream_t st = (cudaStream_t)stream;
  static MgOncePerDevice win_set;  // per device: __constant__ memory belongs to a device
  int dev = 0;
  if (int rc = mg_current_device(&dev, nullptr)) return rc;
  if (!win_set.is_done(dev)) {
    double g[2 * RL_R + 1], sum = 0.0;
    for (int k = 0; k <= 2 * RL_R; k++) { const double x = k - RL_R; g[k] = exp(-(x * x) / (2.0 * 1.5 * 1.5)); sum += g[k]; }
    float w[2 * RL_R + 1];
    for (int k = 0; k <= 2 * RL_R; k++) w[k] = (float)(g[k] / sum);
    MG_CHECK_CUDA(cudaMemcpyToSymbol(c_win, w, sizeof(w)));
    win_set.set_done(dev);
  }
  const size_t n = (size_t)width * height;
  float* d_mu1 = (float*)workspace;
  float* d_e1 = d_mu1 + 3 * n;
  float* d_e12 = d_e1 + 3 * n;
  MG_CHECK_CUDA(cudaMemsetAsync(stats, 0, 3 * sizeof(double), st));
  const dim3 grid((width + RL_T - 1) / RL_T, (height + RL_T - 1) / RL_T, 3), block(RL_T, RL_T);
  ssim_fwd_kernel<<<grid, block, 0, st>>>(width, height, image, target, d_mu1, d_e1, d_e12, stats);
  const double total = 3.0 * (double)n;
  loss_finalize_kernel<<<1, 1, 0, st>>>(stats, total, (double)lambda_dssim);
  ssim_bwd_kernel<<<grid, block, 0, st>>>(width, height, image, target, d_mu1, d_e1, d_e12,
                                          (float)((1.0 - (double)lambda_dssim) / total), (float)((double)lambda_dssim / total), dL_dimage);
  MG_CHECK_LAUNCH();
  return MG_OK;
}
