// renderloss.cu -- mg_render_loss: L_render and dL/dimage on the device.
// Eq. 8 adds lambda_m L_m to "the original rendering loss", which the paper does not define;
// reading 26: the loss of the 3DGS method it modifies,
//     L_render = (1 - lambda) mean|I - G| + lambda (1 - mean SSIM(I, G)),
// SSIM per channel with a separable 11-tap Gaussian window (sigma 1.5), zero padding, C1 = 0.01^2, C2 = 0.03^2.
// Two kernels over 32x32 pixel tiles (+5 pixels of halo staged in shared memory):
//   forward : five filtered maps (I, G, I^2, G^2, IG) -> SSIM, sums of SSIM and |I - G|, and the three partial
//             derivative maps dSSIM/d(mu1, E[I^2], E[IG]);
//   backward: the three maps filtered again (the window is symmetric, so the adjoint is the same filter) and
//             combined with the L1 sign into dL/dI.
// The images are L2-resident at these sizes (13 MB per set of planes), so the kernels are bound by shared-memory loads
// and FMAs, not by HBM.  Both separable passes therefore work from a REGISTER WINDOW: a thread produces 4 consecutive
// outputs from 14 consecutive inputs it loads once (horizontally 3 x LDS.128 + LDS.64 per image row, vertically 14
// conflict-free loads per map), 27 shared-memory loads per output pixel instead of 91 with one output per thread, and
// the 32x32 tile reads 1.72 x its area instead of 2.64 x.  Every tap sum is the same fmaf chain in the same order as a
// plain one-output-per-thread filter (k = 0..10).
#include "mg_common.cuh"

namespace {

constexpr int RL_T = 32;               // tile side
constexpr int RL_R = 5;                // window radius (11 taps)
constexpr int RL_S = RL_T + 2 * RL_R;  // staged side: 42
constexpr int RL_SP = RL_S + 2;        // staged row stride (floats): 44, rows stay 16 B-aligned
constexpr int RL_THREADS = 256;
constexpr int RL_G = RL_T / 4;         // groups of 4 outputs per row / per column: 8
constexpr float RL_C1 = 0.01f * 0.01f, RL_C2 = 0.03f * 0.03f;

__constant__ float c_win[2 * RL_R + 1];

// Stage a (RL_S x RL_S) window of plane `src` around the tile at (x0, y0); zero outside the image.
__device__ __forceinline__ void stage(const float* __restrict__ src, int W, int H, int x0, int y0, float (*dst)[RL_SP]) {
  for (int i = threadIdx.x; i < RL_S * RL_S; i += RL_THREADS) {
    const int r = i / RL_S, c = i - r * RL_S;
    const int y = y0 - RL_R + r, x = x0 - RL_R + c;
    dst[r][c] = (x >= 0 && x < W && y >= 0 && y < H) ? src[(size_t)y * W + x] : 0.f;
  }
}

// 14 consecutive floats of a staged row, starting at a column that is a multiple of 4.
__device__ __forceinline__ void load14(const float* __restrict__ row, float* v) {
  const float4 a = *reinterpret_cast<const float4*>(row), b = *reinterpret_cast<const float4*>(row + 4),
               c = *reinterpret_cast<const float4*>(row + 8);
  const float2 d = *reinterpret_cast<const float2*>(row + 12);
  v[0] = a.x; v[1] = a.y; v[2] = a.z; v[3] = a.w; v[4] = b.x; v[5] = b.y; v[6] = b.z; v[7] = b.w;
  v[8] = c.x; v[9] = c.y; v[10] = c.z; v[11] = c.w; v[12] = d.x; v[13] = d.y;
}

// out[i] = sum_k w[k] v[i + k], i = 0..3, each as one fmaf chain over k = 0..10.
__device__ __forceinline__ void window4(const float* v, float* out) {
#pragma unroll
  for (int i = 0; i < 4; i++) {
    float a = 0.f;
#pragma unroll
    for (int k = 0; k <= 2 * RL_R; k++) a = fmaf(c_win[k], v[i + k], a);
    out[i] = a;
  }
}

__global__ void __launch_bounds__(RL_THREADS) ssim_fwd_kernel(int W, int H, const float* __restrict__ img,
                                                              const float* __restrict__ tgt, float* __restrict__ d_mu1,
                                                              float* __restrict__ d_e1, float* __restrict__ d_e12,
                                                              double* __restrict__ stats) {
  __shared__ __align__(16) float sx[RL_S][RL_SP], sy[RL_S][RL_SP];
  __shared__ __align__(16) float hz[5][RL_S][RL_T];  // horizontally filtered I, G, I^2, G^2, IG
  __shared__ double red[2][RL_THREADS / 32];
  const size_t plane = (size_t)W * H;
  const float* px = img + blockIdx.z * plane;
  const float* py = tgt + blockIdx.z * plane;
  const int x0 = blockIdx.x * RL_T, y0 = blockIdx.y * RL_T;
  stage(px, W, H, x0, y0, sx);
  stage(py, W, H, x0, y0, sy);
  __syncthreads();
  // horizontal pass: task = (staged row r, group g of 4 output columns)
  for (int t = threadIdx.x; t < RL_S * RL_G; t += RL_THREADS) {
    const int r = t / RL_G, g = t - r * RL_G;
    float x[14], y[14], p[14], o[4];
    load14(&sx[r][4 * g], x);
    load14(&sy[r][4 * g], y);
    window4(x, o);
    *reinterpret_cast<float4*>(&hz[0][r][4 * g]) = make_float4(o[0], o[1], o[2], o[3]);
    window4(y, o);
    *reinterpret_cast<float4*>(&hz[1][r][4 * g]) = make_float4(o[0], o[1], o[2], o[3]);
#pragma unroll
    for (int j = 0; j < 14; j++) p[j] = x[j] * x[j];
    window4(p, o);
    *reinterpret_cast<float4*>(&hz[2][r][4 * g]) = make_float4(o[0], o[1], o[2], o[3]);
#pragma unroll
    for (int j = 0; j < 14; j++) p[j] = y[j] * y[j];
    window4(p, o);
    *reinterpret_cast<float4*>(&hz[3][r][4 * g]) = make_float4(o[0], o[1], o[2], o[3]);
#pragma unroll
    for (int j = 0; j < 14; j++) p[j] = x[j] * y[j];
    window4(p, o);
    *reinterpret_cast<float4*>(&hz[4][r][4 * g]) = make_float4(o[0], o[1], o[2], o[3]);
  }
  __syncthreads();
  // vertical pass: thread = (column c, group q of 4 output rows)
  const int c = threadIdx.x & (RL_T - 1), q = threadIdx.x / RL_T;
  float f[5][4];
#pragma unroll
  for (int m = 0; m < 5; m++) {
    float v[14];
#pragma unroll
    for (int j = 0; j < 14; j++) v[j] = hz[m][4 * q + j][c];
    window4(v, f[m]);
  }
  double ssim_d = 0.0, l1_d = 0.0;
  const int x = x0 + c;
#pragma unroll
  for (int i = 0; i < 4; i++) {
    const int y = y0 + 4 * q + i;
    if (x < W && y < H) {
      const float mu1 = f[0][i], mu2 = f[1][i], e1 = f[2][i], e2 = f[3][i], e12 = f[4][i];
      const float s1 = e1 - mu1 * mu1, s2 = e2 - mu2 * mu2, s12 = e12 - mu1 * mu2;
      const float A = 2.f * mu1 * mu2 + RL_C1, B = 2.f * s12 + RL_C2;
      const float C = mu1 * mu1 + mu2 * mu2 + RL_C1, D = s1 + s2 + RL_C2;
      const float iCD = 1.f / (C * D);
      const size_t p = blockIdx.z * plane + (size_t)y * W + x;
      d_mu1[p] = (2.f * mu2 * (B - A)) * iCD - A * B * iCD * iCD * (2.f * mu1 * (D - C));
      d_e1[p] = -A * B * iCD / D;
      d_e12[p] = 2.f * A * iCD;
      ssim_d += (double)(A * B * iCD);
      l1_d += (double)fabsf(sx[4 * q + i + RL_R][c + RL_R] - sy[4 * q + i + RL_R][c + RL_R]);
    }
  }
#pragma unroll
  for (int o = 16; o >= 1; o >>= 1) {
    ssim_d += __shfl_xor_sync(0xffffffffu, ssim_d, o);
    l1_d += __shfl_xor_sync(0xffffffffu, l1_d, o);
  }
  const int t = threadIdx.x;
  if ((t & 31) == 0) { red[0][t >> 5] = l1_d; red[1][t >> 5] = ssim_d; }
  __syncthreads();
  if (t == 0) {
    double a = 0.0, b = 0.0;
#pragma unroll
    for (int w = 0; w < RL_THREADS / 32; w++) { a += red[0][w]; b += red[1][w]; }
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

__global__ void __launch_bounds__(RL_THREADS) ssim_bwd_kernel(int W, int H, const float* __restrict__ img,
                                                              const float* __restrict__ tgt, const float* __restrict__ d_mu1,
                                                              const float* __restrict__ d_e1, const float* __restrict__ d_e12,
                                                              float w_l1, float w_ssim, float* __restrict__ dL_dimage) {
  __shared__ __align__(16) float sm[3][RL_S][RL_SP];
  __shared__ __align__(16) float hz[3][RL_S][RL_T];
  const size_t plane = (size_t)W * H, off = blockIdx.z * plane;
  const int x0 = blockIdx.x * RL_T, y0 = blockIdx.y * RL_T;
  stage(d_mu1 + off, W, H, x0, y0, sm[0]);
  stage(d_e1 + off, W, H, x0, y0, sm[1]);
  stage(d_e12 + off, W, H, x0, y0, sm[2]);
  __syncthreads();
  for (int t = threadIdx.x; t < RL_S * RL_G; t += RL_THREADS) {
    const int r = t / RL_G, g = t - r * RL_G;
#pragma unroll
    for (int m = 0; m < 3; m++) {
      float v[14], o[4];
      load14(&sm[m][r][4 * g], v);
      window4(v, o);
      *reinterpret_cast<float4*>(&hz[m][r][4 * g]) = make_float4(o[0], o[1], o[2], o[3]);
    }
  }
  __syncthreads();
  const int c = threadIdx.x & (RL_T - 1), q = threadIdx.x / RL_T;
  float b[3][4];
#pragma unroll
  for (int m = 0; m < 3; m++) {
    float v[14];
#pragma unroll
    for (int j = 0; j < 14; j++) v[j] = hz[m][4 * q + j][c];
    window4(v, b[m]);
  }
  const int x = x0 + c;
#pragma unroll
  for (int i = 0; i < 4; i++) {
    const int y = y0 + 4 * q + i;
    if (x < W && y < H) {
      const size_t p = off + (size_t)y * W + x;
      const float xi = img[p], yi = tgt[p];
      const float d_ssim = b[0][i] + 2.f * xi * b[1][i] + yi * b[2][i];
      const float sgn = xi > yi ? 1.f : (xi < yi ? -1.f : 0.f);
      dL_dimage[p] = w_l1 * sgn - w_ssim * d_ssim;
    }
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
  const dim3 grid((width + RL_T - 1) / RL_T, (height + RL_T - 1) / RL_T, 3), block(RL_THREADS);
  ssim_fwd_kernel<<<grid, block, 0, st>>>(width, height, image, target, d_mu1, d_e1, d_e12, stats);
  const double total = 3.0 * (double)n;
  loss_finalize_kernel<<<1, 1, 0, st>>>(stats, total, (double)lambda_dssim);
  ssim_bwd_kernel<<<grid, block, 0, st>>>(width, height, image, target, d_mu1, d_e1, d_e12,
                                          (float)((1.0 - (double)lambda_dssim) / total), (float)((double)lambda_dssim / total), dL_dimage);
  MG_CHECK_LAUNCH();
  return MG_OK;
}

// ---- mg_render_loss_static: mg_render_loss for callers that have no way to hand over a workspace.
// Some hosts of this library may not allocate device memory at the point where they need the loss: a renderer or
// trainer embedded in an application whose memory manager took all of the GPU's memory at start-up and hands out only
// the input and output buffers; a plug-in or callback that runs under a "no allocation after initialisation" rule; a
// per-frame loop that must not stall, where cudaMalloc / cudaFree would synchronise the whole device.  For them the
// three derivative maps that the forward kernel leaves for the backward kernel (9 floats per pixel) live in this
// file-scope array, which belongs to the library's image on the device: it is reserved on every GPU that loads this
// part of the library and stays reserved until the process ends (72 MiB at the limit below).
//
// g_rl_scratch is a device symbol.  In host code its name is only a stand-in that the runtime maps to the device
// address; it must never be passed to a kernel as it is.  The address is looked up once per device, with that device
// current, by cudaGetSymbolAddress -- and that look-up is what makes the runtime load this file's kernels and
// reserve the array on the device -- then cached.  After that the call is the existing path, given that address as
// its workspace: the kernels and their arithmetic are the same.
// Nothing in the array has to be zero when a call starts: every element the backward kernel reads (the pixels inside
// the image) was written by the forward kernel of the same call, whatever an earlier call with another image size
// left behind; the three sums are in the caller's `stats`, which the call clears itself.
constexpr size_t RL_STATIC_FLOATS = 9 * (size_t)MG_RENDER_LOSS_STATIC_MAX_PIXELS;
static __device__ __align__(256) float g_rl_scratch[RL_STATIC_FLOATS];

extern "C" int mg_render_loss_static(int32_t width, int32_t height, const float* image, const float* target,
                                     float lambda_dssim, float* dL_dimage, double* stats, void* stream) {
  MG_REQUIRE(width > 0 && height > 0, "image size must be positive");
  const unsigned long long pixels = (unsigned long long)width * (unsigned long long)height;
  if (pixels > (unsigned long long)MG_RENDER_LOSS_STATIC_MAX_PIXELS) {
    mg_set_error("mg_render_loss_static: a %d x %d image has %llu pixels, the built-in scratch holds at most %llu "
                 "(MG_RENDER_LOSS_STATIC_MAX_PIXELS); use mg_render_loss with a workspace of your own",
                 width, height, pixels, (unsigned long long)MG_RENDER_LOSS_STATIC_MAX_PIXELS);
    return MG_ERR_CAPACITY;
  }
  static MgOncePerDevice looked_up;
  static float* address_on[64];  // device address of g_rl_scratch, per device; written before looked_up is set
  int dev = 0;
  if (int rc = mg_current_device(&dev, nullptr)) return rc;
  float* scratch = nullptr;
  if (dev < 64 && looked_up.is_done(dev)) {
    scratch = __atomic_load_n(&address_on[dev], __ATOMIC_RELAXED);
  } else {
    MG_CHECK_CUDA(cudaGetSymbolAddress((void**)&scratch, g_rl_scratch));
    if (scratch == nullptr) {
      mg_set_error("cudaGetSymbolAddress returned a null address for the built-in scratch");
      return MG_ERR_CUDA;
    }
    if (dev < 64) {
      __atomic_store_n(&address_on[dev], scratch, __ATOMIC_RELAXED);
      looked_up.set_done(dev);
    }
  }
  return mg_render_loss(width, height, image, target, lambda_dssim, dL_dimage, stats, scratch,
                        RL_STATIC_FLOATS * sizeof(float), stream);
}
