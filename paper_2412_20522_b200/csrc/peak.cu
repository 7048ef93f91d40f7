// peak.cu -- mg_measure_fp32_peak: the FP32 FMA rate of the device the library runs on, measured, so that the
// roofline of the two blend kernels (plain FP32 arithmetic, no tensor cores) is held against a number timed on
// this chip and not against a product of unit counts ("the bench must measure it").
// Dependent-free FMA chains, every SM busy, CUDA events around >= 50 ms of launches.  Two instruction forms:
// scalar FFMA (one FMA per lane and issue slot) and packed fma.rn.f32x2 (sm_100: two per lane and issue slot).
#include "mg_common.cuh"

namespace {

constexpr int PK_THREADS = 512;
constexpr int PK_CHAINS = 8;    // independent accumulators per thread (latency 4, two issue ports: 8 is enough)
constexpr int PK_UNROLL = 64;   // FMA rounds per loop iteration

__global__ void __launch_bounds__(PK_THREADS) fma_scalar_kernel(int iters, float a, float b, float* __restrict__ sink) {
  float x[PK_CHAINS];
#pragma unroll
  for (int c = 0; c < PK_CHAINS; c++) x[c] = (float)(threadIdx.x + c) * 1e-3f;
  for (int it = 0; it < iters; it++) {
#pragma unroll
    for (int u = 0; u < PK_UNROLL; u++) {
#pragma unroll
      for (int c = 0; c < PK_CHAINS; c++) x[c] = fmaf(x[c], a, b);
    }
  }
  float s = 0.f;
#pragma unroll
  for (int c = 0; c < PK_CHAINS; c++) s += x[c];
  if (s == 123.456f) sink[0] = s;  // never true for the constants used; keeps the chains alive
}

__global__ void __launch_bounds__(PK_THREADS) fma_packed_kernel(int iters, float a, float b, float* __restrict__ sink) {
  float2 x[PK_CHAINS];
  const float2 a2 = make_float2(a, a), b2 = make_float2(b, b);
#pragma unroll
  for (int c = 0; c < PK_CHAINS; c++) x[c] = make_float2((float)(threadIdx.x + c) * 1e-3f, (float)c * 1e-3f);
  for (int it = 0; it < iters; it++) {
#pragma unroll
    for (int u = 0; u < PK_UNROLL; u++) {
#pragma unroll
      for (int c = 0; c < PK_CHAINS; c++) x[c] = __ffma2_rn(x[c], a2, b2);
    }
  }
  float s = 0.f;
#pragma unroll
  for (int c = 0; c < PK_CHAINS; c++) s += x[c].x + x[c].y;
  if (s == 123.456f) sink[0] = s;
}

}  // namespace

extern "C" int mg_measure_fp32_peak(double min_seconds, double* tflops_host, float* scratch, void* stream) {
  MG_REQUIRE(scratch != nullptr && tflops_host != nullptr, "scratch (one device float) or tflops_host (4 doubles) is null");
  MG_REQUIRE(min_seconds >= 0.0 && min_seconds <= 10.0, "min_seconds must be in [0, 10]");
  int sms = 0;
  if (int rc = mg_current_device(nullptr, &sms)) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  struct Events {  // destroyed on every way out, the MG_CHECK_CUDA early returns included
    cudaEvent_t a = nullptr, b = nullptr;
    ~Events() {
      if (a) cudaEventDestroy(a);
      if (b) cudaEventDestroy(b);
    }
  } ev;
  MG_CHECK_CUDA(cudaEventCreate(&ev.a));
  MG_CHECK_CUDA(cudaEventCreate(&ev.b));
  const cudaEvent_t e0 = ev.a, e1 = ev.b;
  const int grid = sms * 4;  // 4 blocks of 512 threads per SM: every warp slot taken
  const int iters = 256;
  for (int form = 0; form < 2; form++) {
    const double flop_per_launch = 2.0 * (form + 1) * PK_CHAINS * PK_UNROLL * (double)iters * PK_THREADS * grid;
    double best = 0.0, spent = 0.0, flop = 0.0;
    const int reps = 4;
    for (int round = 0; round < 64 && (round < 2 || spent < min_seconds); round++) {
      MG_CHECK_CUDA(cudaEventRecord(e0, st));
      for (int r = 0; r < reps; r++) {
        if (form == 0) fma_scalar_kernel<<<grid, PK_THREADS, 0, st>>>(iters, 0.999f, 1e-3f, scratch);
        else fma_packed_kernel<<<grid, PK_THREADS, 0, st>>>(iters, 0.999f, 1e-3f, scratch);
      }
      MG_CHECK_CUDA(cudaEventRecord(e1, st));
      MG_CHECK_CUDA(cudaEventSynchronize(e1));
      MG_CHECK_LAUNCH();
      float ms = 0.f;
      MG_CHECK_CUDA(cudaEventElapsedTime(&ms, e0, e1));
      const double sec = ms * 1e-3;
      if (round > 0) {  // round 0 warms up
        spent += sec;
        flop += flop_per_launch * reps;
        const double tf = flop_per_launch * reps / sec / 1e12;
        if (tf > best) best = tf;
      }
    }
    tflops_host[2 * form] = flop / spent / 1e12;  // sustained over the whole measurement
    tflops_host[2 * form + 1] = best;             // best round (burst)
  }
  return MG_OK;
}
