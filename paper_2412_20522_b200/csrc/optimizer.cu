// optimizer.cu -- density-control statistics and the optimiser step (readings 27-28).
//   mg_density_stats  per visible Gaussian: grad_accum += |(sx, sy) . dL/dmean2d|, denom += 1, max_radii = max(., radius)
//   mg_adam_step      Adam with bias correction over up to 8 attribute groups (own learning rate each) in ONE launch
// The paper keeps "the densification scheme" and the training procedure of the method it modifies
// and prints neither; the readings say what is computed.  Both are elementwise and HBM-bound: 28 B per parameter float
// (read p, g, m, v; write p, m, v), 128-bit accesses, four independent vectors in flight per thread.
#include "mg_common.cuh"

namespace {

constexpr int OP_THREADS = 256;
constexpr int OP_VEC_PER_THREAD = 4;
constexpr int OP_FLOATS_PER_BLOCK = OP_THREADS * OP_VEC_PER_THREAD * 4;

struct AdamGroupDev {
  float* p;
  const float* g;
  float* m;
  float* v;
  unsigned long long total;  // floats
  unsigned int row_floats;
  float step_size;           // lr / (1 - beta1^t)
  unsigned int block_begin;  // first block of this group
  unsigned int rf_magic;     // ceil(2^32 / row_floats) (0 if row_floats == 1): floor(x / row_floats) = umulhi(x, magic) for x < 2^16
};
struct AdamParams {
  AdamGroupDev grp[MG_ADAM_MAX_GROUPS];
  int n_groups;
  float b1, one_minus_b1, b2, one_minus_b2, inv_sqrt_bc2, eps;  // inv_sqrt_bc2 = 1 / sqrt(1 - beta2^t)
};

__device__ __forceinline__ void adam_one(float& p, float g, float& m, float& v, const AdamParams& P, float step_size) {
  m = fmaf(P.b1, m, P.one_minus_b1 * g);
  v = fmaf(P.b2, v, P.one_minus_b2 * g * g);
  const float denom = fmaf(sqrtf(v), P.inv_sqrt_bc2, P.eps);
  p = p - step_size * m / denom;
}

// kRows: radii given -> rows of Gaussians with radius 0 are neither read (beyond the radius) nor written.
template <bool kRows>
__global__ void __launch_bounds__(OP_THREADS) adam_kernel(const __grid_constant__ AdamParams P, const int32_t* __restrict__ radii) {
  int gi = 0;
#pragma unroll
  for (int i = 1; i < MG_ADAM_MAX_GROUPS; i++)
    if (i < P.n_groups && blockIdx.x >= P.grp[i].block_begin) gi = i;
  const AdamGroupDev& G = P.grp[gi];
  const unsigned long long base = (unsigned long long)(blockIdx.x - G.block_begin) * OP_FLOATS_PER_BLOCK;
  const float step_size = G.step_size;
  // Row of an element (kRows): ONE division per block -- the block's first element is base = row0 * row_floats + rem0 --
  // and from there the in-block offset x = rem0 + (element - base) < 4096 + 1024 is divided by a multiply-high with the
  // host's reciprocal, exact for x row_floats < 2^32.  When row_floats is a multiple of 4 a vector lies within one row.
  const unsigned int rf = G.row_floats, magic = G.rf_magic;
  const unsigned long long row0 = kRows ? base / rf : 0ull;
  const unsigned int rem0 = kRows ? (unsigned int)(base - row0 * rf) : 0u;
  const bool vec_in_row = (rf & 3u) == 0u;

  unsigned long long e[OP_VEC_PER_THREAD];
  unsigned int vis[OP_VEC_PER_THREAD];  // bit j: element e + j is to be updated
#pragma unroll
  for (int k = 0; k < OP_VEC_PER_THREAD; k++) {
    e[k] = base + 4ull * (k * OP_THREADS + threadIdx.x);
    vis[k] = 0;
    if (e[k] < G.total) {
      const unsigned int nvalid = (unsigned int)min(4ull, G.total - e[k]);
      vis[k] = (1u << nvalid) - 1u;
      if (kRows) {
        const unsigned int x = rem0 + 4u * (unsigned int)(k * OP_THREADS + threadIdx.x);
        unsigned int mbits = 0;
        if (vec_in_row) {
          if (radii[row0 + __umulhi(x, magic)] > 0) mbits = vis[k];
        } else {
#pragma unroll
          for (unsigned int j = 0; j < 4; j++) {
            if (j < nvalid) {
              const unsigned int r = magic ? __umulhi(x + j, magic) : x + j;
              if (radii[row0 + r] > 0) mbits |= 1u << j;
            }
          }
        }
        vis[k] = mbits;
      }
    }
  }
  float4 p[OP_VEC_PER_THREAD], g[OP_VEC_PER_THREAD], m[OP_VEC_PER_THREAD], v[OP_VEC_PER_THREAD];
  // every group's arrays are 16-byte aligned (mg.h) and e is a multiple of 4: a vector whose 4 elements exist is aligned
#pragma unroll
  for (int k = 0; k < OP_VEC_PER_THREAD; k++) {
    if (vis[k] && e[k] + 4 <= G.total) {
      p[k] = *reinterpret_cast<const float4*>(G.p + e[k]);
      g[k] = __ldg(reinterpret_cast<const float4*>(G.g + e[k]));
      m[k] = *reinterpret_cast<const float4*>(G.m + e[k]);
      v[k] = *reinterpret_cast<const float4*>(G.v + e[k]);
    }
  }
#pragma unroll
  for (int k = 0; k < OP_VEC_PER_THREAD; k++) {
    if (!vis[k]) continue;
    if (e[k] + 4 <= G.total) {
      float4 pn = p[k], mn = m[k], vn = v[k];
      adam_one(pn.x, g[k].x, mn.x, vn.x, P, step_size);
      adam_one(pn.y, g[k].y, mn.y, vn.y, P, step_size);
      adam_one(pn.z, g[k].z, mn.z, vn.z, P, step_size);
      adam_one(pn.w, g[k].w, mn.w, vn.w, P, step_size);
      if (kRows && vis[k] != 0xfu) {  // the vector straddles a row that is not updated: only the updated floats are
        const float pa[4] = {pn.x, pn.y, pn.z, pn.w}, ma[4] = {mn.x, mn.y, mn.z, mn.w}, va[4] = {vn.x, vn.y, vn.z, vn.w};
#pragma unroll
        for (unsigned int j = 0; j < 4; j++) {  // stored, so that a skipped row is really not written (include/mg.h)
          if ((vis[k] >> j) & 1u) {
            G.p[e[k] + j] = pa[j]; G.m[e[k] + j] = ma[j]; G.v[e[k] + j] = va[j];
          }
        }
        continue;
      }
      *reinterpret_cast<float4*>(G.p + e[k]) = pn;
      *reinterpret_cast<float4*>(G.m + e[k]) = mn;
      *reinterpret_cast<float4*>(G.v + e[k]) = vn;
    } else {  // ragged tail of the group: at most 3 floats
      for (unsigned int j = 0; j < 4; j++) {
        if ((vis[k] >> j) & 1u) {
          const unsigned long long i = e[k] + j;
          float pj = G.p[i], mj = G.m[i], vj = G.v[i];
          adam_one(pj, G.g[i], mj, vj, P, step_size);
          G.p[i] = pj; G.m[i] = mj; G.v[i] = vj;
        }
      }
    }
  }
}

__global__ void __launch_bounds__(OP_THREADS) density_stats_kernel(int64_t N, const float2* __restrict__ dL_dmeans2d,
                                                                   const int32_t* __restrict__ radii, float sx, float sy,
                                                                   float* __restrict__ grad_accum, float* __restrict__ denom,
                                                                   float* __restrict__ max_radii) {
  const int64_t i = (int64_t)blockIdx.x * OP_THREADS + threadIdx.x;
  if (i >= N) return;
  const int32_t r = radii[i];
  if (r <= 0) return;  // not visible in this view: nothing is read or written
  const float2 g = __ldg(dL_dmeans2d + i);
  const float gx = sx * g.x, gy = sy * g.y;
  grad_accum[i] += sqrtf(fmaf(gx, gx, gy * gy));
  denom[i] += 1.f;
  max_radii[i] = fmaxf(max_radii[i], (float)r);
}

}  // namespace

extern "C" int mg_density_stats(int64_t N, const float* dL_dmeans2d, const int32_t* radii, float scale_x, float scale_y,
                                float* grad_accum, float* denom, float* max_radii, void* stream) {
  MG_REQUIRE(N >= 0 && N < (int64_t)1 << 31, "N must be in [0, 2^31)");
  if (N == 0) return MG_OK;
  MG_REQUIRE(dL_dmeans2d && radii && grad_accum && denom && max_radii, "null array");
  density_stats_kernel<<<(unsigned)((N + OP_THREADS - 1) / OP_THREADS), OP_THREADS, 0, (cudaStream_t)stream>>>(
      N, (const float2*)dL_dmeans2d, radii, scale_x, scale_y, grad_accum, denom, max_radii);
  MG_CHECK_LAUNCH();
  return MG_OK;
}

extern "C" int mg_adam_step(int32_t n_groups, const mg_adam_group* groups_host, float beta1, float beta2, float eps,
                            int64_t step, const int32_t* radii, void* stream) {
  MG_REQUIRE(n_groups >= 0 && n_groups <= MG_ADAM_MAX_GROUPS, "n_groups must be in [0, MG_ADAM_MAX_GROUPS]");
  MG_REQUIRE(n_groups == 0 || groups_host, "groups_host is null");
  MG_REQUIRE(step >= 1, "step counts from 1");
  MG_REQUIRE(beta1 >= 0.f && beta1 < 1.f && beta2 >= 0.f && beta2 < 1.f && eps >= 0.f, "beta1, beta2 in [0,1), eps >= 0");
  AdamParams P;
  P.n_groups = 0;
  const double bc1 = 1.0 - pow((double)beta1, (double)step), bc2 = 1.0 - pow((double)beta2, (double)step);
  P.b1 = beta1; P.one_minus_b1 = (float)(1.0 - (double)beta1);
  P.b2 = beta2; P.one_minus_b2 = (float)(1.0 - (double)beta2);
  P.inv_sqrt_bc2 = (float)(1.0 / sqrt(bc2));
  P.eps = eps;
  unsigned long long blocks = 0;
  int64_t rows0 = -1;
  for (int i = 0; i < n_groups; i++) {
    const mg_adam_group& g = groups_host[i];
    MG_REQUIRE(g.n_rows >= 0 && g.n_rows < (int64_t)1 << 31 && g.row_floats >= 1 && g.row_floats <= 1024, "group shape");
    if (radii) {
      MG_REQUIRE(rows0 < 0 || rows0 == g.n_rows, "with radii every group must have one row per Gaussian");
      rows0 = g.n_rows;
    }
    if (g.n_rows == 0) continue;
    MG_REQUIRE(g.param && g.grad && g.m && g.v, "null array in a group");
    MG_REQUIRE((((uintptr_t)g.param | (uintptr_t)g.grad | (uintptr_t)g.m | (uintptr_t)g.v) & 15) == 0, "arrays must be 16-byte aligned");
    AdamGroupDev& d = P.grp[P.n_groups++];
    d.p = g.param; d.g = g.grad; d.m = g.m; d.v = g.v;
    d.total = (unsigned long long)g.n_rows * (unsigned long long)g.row_floats;
    d.row_floats = (unsigned int)g.row_floats;
    d.rf_magic = g.row_floats == 1 ? 0u : (unsigned int)(((1ull << 32) + (unsigned long long)g.row_floats - 1) / (unsigned long long)g.row_floats);
    d.step_size = (float)((double)g.lr / bc1);
    d.block_begin = (unsigned int)blocks;
    blocks += (d.total + OP_FLOATS_PER_BLOCK - 1) / OP_FLOATS_PER_BLOCK;
    MG_REQUIRE(blocks < (1ull << 31), "too many parameters for one launch");
  }
  if (blocks == 0) return MG_OK;
  if (radii)
    adam_kernel<true><<<(unsigned)blocks, OP_THREADS, 0, (cudaStream_t)stream>>>(P, radii);
  else
    adam_kernel<false><<<(unsigned)blocks, OP_THREADS, 0, (cudaStream_t)stream>>>(P, nullptr);
  MG_CHECK_LAUNCH();
  return MG_OK;
}
