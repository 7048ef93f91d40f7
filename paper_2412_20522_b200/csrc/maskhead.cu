// maskhead.cu -- the mask head around the rasterizer.
//   mg_mask_sample      Gumbel-Softmax over 2 scores per Gaussian -> hard mask M_i in {0,1} + soft sample
//   mg_mask_sample_bwd  straight-through gradient of the sample to the two scores
//   mg_mask_loss        lambda_m L_m = lambda_m (mean M)^2 (Eq. 7-8) and its gradient, added to dL/dM
//   mg_mask_prune_keep  "sample each Gaussian 10 times and remove those that are never sampled"
//   mg_compact          stable compaction of the attribute arrays by the keep flags
// All elementwise and HBM-bound: one pass over the data, coalesced, no intermediate arrays.  Random numbers are
// inputs (uniforms in (0,1)); the library draws none.
#include <cooperative_groups.h>

#include "mg_common.cuh"

namespace cg = cooperative_groups;

namespace {

constexpr int MH_THREADS = 256;
constexpr int ML_BLOCKS_PER_SM = 4;  // mg_mask_loss: grid = at most this many blocks per SM (and never more than can be resident)

// d = (s_1 + g_1) - (s_0 + g_0) with g = -log(-log u): the hard sample is d > 0, the soft one sigmoid(d / tau).
// A uniform outside (0,1) is taken as the nearest fp32 value inside it (include/mg.h, reading 29): the noise
// stays within [-4.47, 16.64] and d is finite whatever the caller's generator returns at its endpoints.
__device__ __forceinline__ float perturbed_gap(float2 s, float2 u) {
  u.x = fminf(fmaxf(u.x, 1.17549435e-38f), 0.99999994f);
  u.y = fminf(fmaxf(u.y, 1.17549435e-38f), 0.99999994f);
  // inner log accurate (for u near 1, -log u is tiny and needs its relative accuracy), outer log lg2-based
  const float g0 = -__logf(-logf(u.x)), g1 = -__logf(-logf(u.y));
  return (s.y + g1) - (s.x + g0);
}

__global__ void __launch_bounds__(MH_THREADS) mask_sample_kernel(int64_t N, const float2* __restrict__ scores,
                                                                 const float2* __restrict__ uniforms, float inv_tau,
                                                                 float* __restrict__ masks, float* __restrict__ soft) {
  const int64_t i = (int64_t)blockIdx.x * MH_THREADS + threadIdx.x;
  if (i >= N) return;
  const float d = perturbed_gap(scores[i], uniforms[i]);
  masks[i] = d > 0.f ? 1.f : 0.f;
  if (soft) soft[i] = 1.f / (1.f + expf(-d * inv_tau));
}

__global__ void __launch_bounds__(MH_THREADS) mask_sample_bwd_kernel(int64_t N, const float* __restrict__ soft,
                                                                     const float* __restrict__ dL_dmask, float inv_tau,
                                                                     float2* __restrict__ dL_dscores) {
  const int64_t i = (int64_t)blockIdx.x * MH_THREADS + threadIdx.x;
  if (i >= N) return;
  const float y = soft[i];
  const float t = dL_dmask[i] * y * (1.f - y) * inv_tau;
  dL_dscores[i] = make_float2(-t, t);
}

// stats[0] += sum of masks (double: exact for 0/1 masks whatever the order of the atomics)
// L_m and its gradient in ONE kernel (two launches in round 1).  Every element needs the mean over all of them, so the
// grid meets once: phase 1 sums the masks into stats[0]; grid.sync(); phase 2 adds lambda_m 2 mean / N to dL_dmask and
// block 0 writes the two results.  The barrier is the cooperative-groups one (the launch is cooperative, so the runtime
// refuses a grid that could not be resident at once); it keeps its state outside the caller's arrays.  The grid is a few
// blocks per SM, not the whole GPU: a 12 MB read needs no more, and the rest of the GPU stays free for work on other
// streams.  Both phases move float4s (masks and dL_dmask are 16-byte aligned, include/mg.h), the tail singly.
__global__ void __launch_bounds__(MH_THREADS) mask_loss_kernel(int64_t N, const float* __restrict__ masks, double lambda_m,
                                                               float* __restrict__ dL_dmask, double* __restrict__ stats) {
  __shared__ double part[MH_THREADS / 32];
  const int64_t stride = (int64_t)gridDim.x * MH_THREADS, first = (int64_t)blockIdx.x * MH_THREADS + threadIdx.x;
  const int64_t n4 = N >> 2;
  const float4* __restrict__ masks4 = reinterpret_cast<const float4*>(masks);
  double s = 0.0;
  for (int64_t i = first; i < n4; i += stride) {
    const float4 v = masks4[i];
    s += ((double)v.x + (double)v.y) + ((double)v.z + (double)v.w);
  }
  for (int64_t i = 4 * n4 + first; i < N; i += stride) s += (double)masks[i];
#pragma unroll
  for (int o = 16; o >= 1; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
  if ((threadIdx.x & 31) == 0) part[threadIdx.x >> 5] = s;
  __syncthreads();
  if (threadIdx.x == 0) {
    double t = 0.0;
#pragma unroll
    for (int w = 0; w < MH_THREADS / 32; w++) t += part[w];
    if (t != 0.0) atomicAdd(&stats[0], t);
  }
  cg::this_grid().sync();
  const double mean = *reinterpret_cast<volatile double*>(&stats[0]) / (double)N;
  if (dL_dmask) {
    const float add = (float)(lambda_m * 2.0 * mean / (double)N);
    float4* __restrict__ g4 = reinterpret_cast<float4*>(dL_dmask);
    for (int64_t i = first; i < n4; i += stride) {
      float4 v = g4[i];
      v.x += add; v.y += add; v.z += add; v.w += add;
      g4[i] = v;
    }
    for (int64_t i = 4 * n4 + first; i < N; i += stride) dL_dmask[i] += add;
  }
  if (blockIdx.x == 0 && threadIdx.x == 0) {
    stats[1] = lambda_m * mean * mean;
    stats[2] = mean;
  }
}

__global__ void __launch_bounds__(MH_THREADS) mask_prune_kernel(int64_t N, int S, const float2* __restrict__ scores,
                                                                const float2* __restrict__ uniforms, uint8_t* __restrict__ keep) {
  const int64_t i = (int64_t)blockIdx.x * MH_THREADS + threadIdx.x;
  if (i >= N) return;
  const float2 s = scores[i];
  bool k = false;
  for (int d = 0; d < S; d++) k = k || perturbed_gap(s, uniforms[(int64_t)d * N + i]) > 0.f;
  keep[i] = k ? 1 : 0;
}

// ---- compaction: block counts -> scan of the block counts (one block) -> positions -> row copies
constexpr int CP_BLOCK = 1024;

__global__ void __launch_bounds__(CP_BLOCK) compact_count_kernel(int64_t N, const uint8_t* __restrict__ keep, uint32_t* __restrict__ block_counts) {
  const int64_t i = (int64_t)blockIdx.x * CP_BLOCK + threadIdx.x;
  const int c = __syncthreads_count(i < N && keep[i] != 0);
  if (threadIdx.x == 0) block_counts[blockIdx.x] = (uint32_t)c;
}

__global__ void __launch_bounds__(1024) compact_scan_kernel(uint32_t* __restrict__ block_counts, int nblk, unsigned long long* __restrict__ total) {
  __shared__ uint32_t part[1024];
  const int per = (nblk + 1023) / 1024;
  const int b = threadIdx.x * per, e = min(nblk, b + per);
  uint32_t s = 0;
  for (int j = b; j < e; j++) s += block_counts[j];
  part[threadIdx.x] = s;
  __syncthreads();
  for (int o = 1; o < 1024; o <<= 1) {
    const uint32_t v = threadIdx.x >= o ? part[threadIdx.x - o] : 0;
    __syncthreads();
    part[threadIdx.x] += v;
    __syncthreads();
  }
  uint32_t run = part[threadIdx.x] - s;
  for (int j = b; j < e; j++) { const uint32_t v = block_counts[j]; block_counts[j] = run; run += v; }
  if (threadIdx.x == 1023) *total = part[1023];
}

__global__ void __launch_bounds__(CP_BLOCK) compact_pos_kernel(int64_t N, const uint8_t* __restrict__ keep,
                                                               const uint32_t* __restrict__ block_offsets, uint32_t* __restrict__ pos) {
  __shared__ uint32_t wsum[CP_BLOCK / 32];
  const int64_t i = (int64_t)blockIdx.x * CP_BLOCK + threadIdx.x;
  const bool k = i < N && keep[i] != 0;
  const uint32_t ballot = __ballot_sync(0xffffffffu, k);
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  if (lane == 0) wsum[warp] = __popc(ballot);
  __syncthreads();
  uint32_t woff = 0;
  for (int w = 0; w < warp; w++) woff += wsum[w];
  if (i < N) pos[i] = k ? block_offsets[blockIdx.x] + woff + __popc(ballot & ((1u << lane) - 1u)) : 0xffffffffu;
}

// Input elements (a float, or a float4 when the row size is a multiple of 4 floats): element e of an array with r
// elements per row belongs to Gaussian e / r.  CP_PER elements per thread, a block apart, all their loads issued before
// any is stored (a copy is bound by the bytes in flight).  kR > 0: the row size is a compile-time constant, so the
// division is a multiply (the sizes this method has: 1, 2, 3 and 12 elements per row); kR == 0: any r, a runtime
// division.  32-bit index arithmetic (the host checks the range).
constexpr int CP_PER = 4;
template <typename V, int kR>
__global__ void __launch_bounds__(MH_THREADS) compact_rows_kernel(uint32_t n_elems, uint32_t r_rt, const uint32_t* __restrict__ pos,
                                                                  const V* __restrict__ src, V* __restrict__ dst) {
  const uint32_t r = kR > 0 ? (uint32_t)kR : r_rt;
  const uint32_t e0 = blockIdx.x * (uint32_t)(MH_THREADS * CP_PER) + threadIdx.x;
  uint32_t p[CP_PER], j[CP_PER];
#pragma unroll
  for (int q = 0; q < CP_PER; q++) {
    const uint32_t e = e0 + q * MH_THREADS;
    p[q] = 0xffffffffu;
    j[q] = 0;
    if (e < n_elems) {
      const uint32_t i = e / r;
      j[q] = e - i * r;
      p[q] = pos[i];
    }
  }
  V v[CP_PER];
#pragma unroll
  for (int q = 0; q < CP_PER; q++)
    if (p[q] != 0xffffffffu) v[q] = src[e0 + q * MH_THREADS];
#pragma unroll
  for (int q = 0; q < CP_PER; q++)
    if (p[q] != 0xffffffffu) dst[(size_t)p[q] * r + j[q]] = v[q];
}

template <typename V>
void compact_rows_launch(uint32_t ne, uint32_t r, const uint32_t* pos, const V* src, V* dst, cudaStream_t st) {
  const unsigned grid = (unsigned)(((uint64_t)ne + MH_THREADS * CP_PER - 1) / (MH_THREADS * CP_PER));
  switch (r) {
    case 1: compact_rows_kernel<V, 1><<<grid, MH_THREADS, 0, st>>>(ne, r, pos, src, dst); break;
    case 2: compact_rows_kernel<V, 2><<<grid, MH_THREADS, 0, st>>>(ne, r, pos, src, dst); break;
    case 3: compact_rows_kernel<V, 3><<<grid, MH_THREADS, 0, st>>>(ne, r, pos, src, dst); break;
    case 12: compact_rows_kernel<V, 12><<<grid, MH_THREADS, 0, st>>>(ne, r, pos, src, dst); break;
    default: compact_rows_kernel<V, 0><<<grid, MH_THREADS, 0, st>>>(ne, r, pos, src, dst); break;
  }
}

inline size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }

}  // namespace

extern "C" int mg_mask_sample(int64_t N, const float* scores, const float* uniforms, float tau, float* masks, float* soft,
                              void* stream) {
  MG_REQUIRE(N >= 0 && N < (int64_t)1 << 31, "N must be in [0, 2^31)");
  MG_REQUIRE(tau > 0.f, "tau must be positive");
  if (N == 0) return MG_OK;
  MG_REQUIRE(scores && uniforms && masks, "null array");
  mask_sample_kernel<<<(unsigned)((N + MH_THREADS - 1) / MH_THREADS), MH_THREADS, 0, (cudaStream_t)stream>>>(
      N, (const float2*)scores, (const float2*)uniforms, 1.f / tau, masks, soft);
  MG_CHECK_LAUNCH();
  return MG_OK;
}

extern "C" int mg_mask_sample_bwd(int64_t N, const float* soft, const float* dL_dmask, float tau, float* dL_dscores,
                                  void* stream) {
  MG_REQUIRE(N >= 0 && N < (int64_t)1 << 31, "N must be in [0, 2^31)");
  MG_REQUIRE(tau > 0.f, "tau must be positive");
  if (N == 0) return MG_OK;
  MG_REQUIRE(soft && dL_dmask && dL_dscores, "null array");
  mask_sample_bwd_kernel<<<(unsigned)((N + MH_THREADS - 1) / MH_THREADS), MH_THREADS, 0, (cudaStream_t)stream>>>(
      N, soft, dL_dmask, 1.f / tau, (float2*)dL_dscores);
  MG_CHECK_LAUNCH();
  return MG_OK;
}

extern "C" int mg_mask_loss(int64_t N, const float* masks, float lambda_m, float* dL_dmask, double* stats, void* stream) {
  MG_REQUIRE(N > 0 && N < (int64_t)1 << 31, "N must be in (0, 2^31)");
  MG_REQUIRE(masks && stats, "null array");
  cudaStream_t st = (cudaStream_t)stream;
  MG_CHECK_CUDA(cudaMemsetAsync(stats, 0, 3 * sizeof(double), st));
  const int64_t want = (N / 4 + MH_THREADS - 1) / MH_THREADS + 1;
  static MgOncePerDevice asked;   // the occupancy query costs as much host time as the kernel runs: once per device
  static int per_sm_of[64];
  int dev = 0, sms = 0, per_sm = 0;
  if (int rc = mg_current_device(&dev, &sms)) return rc;
  if (dev < 64 && asked.is_done(dev)) {
    per_sm = __atomic_load_n(&per_sm_of[dev], __ATOMIC_RELAXED);
  } else {
    MG_CHECK_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, mask_loss_kernel, MH_THREADS, 0));
    if (per_sm < 1) per_sm = 1;
    if (dev < 64) {
      __atomic_store_n(&per_sm_of[dev], per_sm, __ATOMIC_RELAXED);
      asked.set_done(dev);
    }
  }
  const int64_t resident = (int64_t)sms * (per_sm < ML_BLOCKS_PER_SM ? per_sm : ML_BLOCKS_PER_SM);
  const unsigned grid = (unsigned)(want < resident ? want : resident);
  double lam = (double)lambda_m;
  void* args[] = {(void*)&N, (void*)&masks, (void*)&lam, (void*)&dL_dmask, (void*)&stats};
  MG_CHECK_CUDA(cudaLaunchCooperativeKernel((const void*)mask_loss_kernel, dim3(grid), dim3(MH_THREADS), args, 0, st));
  return MG_OK;
}

extern "C" int mg_mask_prune_keep(int64_t N, int32_t n_draws, const float* scores, const float* uniforms, uint8_t* keep,
                                  void* stream) {
  MG_REQUIRE(N >= 0 && N < (int64_t)1 << 31, "N must be in [0, 2^31)");
  MG_REQUIRE(n_draws >= 0, "n_draws must be >= 0");
  if (N == 0) return MG_OK;
  MG_REQUIRE(scores && keep && (uniforms || n_draws == 0), "null array");
  mask_prune_kernel<<<(unsigned)((N + MH_THREADS - 1) / MH_THREADS), MH_THREADS, 0, (cudaStream_t)stream>>>(
      N, n_draws, (const float2*)scores, (const float2*)uniforms, keep);
  MG_CHECK_LAUNCH();
  return MG_OK;
}

extern "C" size_t mg_compact_workspace_bytes(int64_t N) {
  if (N < 0) return 0;
  const size_t nblk = (size_t)((N + CP_BLOCK - 1) / CP_BLOCK);
  return align256(8) + align256(4 * (nblk + 1)) + align256(4 * (size_t)N);
}

extern "C" int mg_compact(int64_t N, const uint8_t* keep, int32_t n_arrays, const float* const* src, float* const* dst,
                          const int32_t* row_floats, void* workspace, size_t workspace_bytes, uint64_t* N_out_host,
                          void* stream) {
  MG_REQUIRE(N >= 0 && N < (int64_t)1 << 31, "N must be in [0, 2^31)");
  MG_REQUIRE(n_arrays >= 0 && n_arrays <= 16, "n_arrays must be in 0..16");
  MG_REQUIRE(workspace != nullptr && ((uintptr_t)workspace & 255) == 0, "workspace must be non-null and 256-byte aligned");
  if (workspace_bytes < mg_compact_workspace_bytes(N)) {
    mg_set_error("workspace too small: %zu bytes given, %zu needed", workspace_bytes, mg_compact_workspace_bytes(N));
    return MG_ERR_CAPACITY;
  }
  cudaStream_t st = (cudaStream_t)stream;
  char* ws = (char*)workspace;
  unsigned long long* total = (unsigned long long*)ws;
  const int nblk = (int)((N + CP_BLOCK - 1) / CP_BLOCK);
  uint32_t* block_counts = (uint32_t*)(ws + align256(8));
  uint32_t* pos = (uint32_t*)(ws + align256(8) + align256(4 * ((size_t)nblk + 1)));
  MG_CHECK_CUDA(cudaMemsetAsync(total, 0, 8, st));
  if (N > 0) {
    MG_REQUIRE(keep && (n_arrays == 0 || (src && dst && row_floats)), "null array");
    compact_count_kernel<<<nblk, CP_BLOCK, 0, st>>>(N, keep, block_counts);
    compact_scan_kernel<<<1, 1024, 0, st>>>(block_counts, nblk, total);
    compact_pos_kernel<<<nblk, CP_BLOCK, 0, st>>>(N, keep, block_counts, pos);
    for (int a = 0; a < n_arrays; a++) {
      MG_REQUIRE(src[a] && dst[a] && row_floats[a] > 0, "null array or non-positive row size");
      const bool vec = row_floats[a] % 4 == 0 && ((uintptr_t)src[a] & 15) == 0 && ((uintptr_t)dst[a] & 15) == 0;
      const int64_t r = vec ? row_floats[a] / 4 : row_floats[a];
      const int64_t ne = N * r;
      MG_REQUIRE(ne < ((int64_t)1 << 32) - MH_THREADS * CP_PER, "array too large for one compaction call (N * row size >= 2^32 elements)");
      if (vec) compact_rows_launch<float4>((uint32_t)ne, (uint32_t)r, pos, (const float4*)src[a], (float4*)dst[a], st);
      else compact_rows_launch<float>((uint32_t)ne, (uint32_t)r, pos, src[a], dst[a], st);
    }
    MG_CHECK_LAUNCH();
  }
  if (N_out_host) MG_CHECK_CUDA(cudaMemcpyAsync(N_out_host, total, sizeof(uint64_t), cudaMemcpyDeviceToHost, st));
  return MG_OK;
}
