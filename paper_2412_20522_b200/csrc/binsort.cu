// binsort.cu -- mg_bin_sort: key duplication, (tile, depth) radix sort, tile ranges.
// Steps a4-a6 of the hot path (PAPER.md:66 "depth order", :74 16x16 tiles; O9).
//
// The result is the ascending order of the 64-bit keys (tile_id << 32 | depth bits), ties by index.
// It is produced by an LSD radix sort of that key whose four depth-digit passes are HOISTED BEFORE
// the key duplication: all duplicates of a Gaussian share its depth, so sorting the N Gaussians by
// depth first (stable, 4 x 8 bits) and emitting the duplicates in that order leaves only the
// ceil(log2(tiles)) tile bits to sort over the R duplicated keys (2 stable passes for <= 65536
// tiles).  Per duplicated key this moves ~44 B instead of ~150 B for six 64-bit key-value passes.
// Tile ranges come from a summed-area table of the tile rectangles (4 atomics per Gaussian), not
// from a pass over the sorted keys.
#include "mg_common.cuh"

namespace {

constexpr int RS_THREADS = 512;
constexpr int RS_ITEMS = 16;
constexpr int RS_WARPS = RS_THREADS / 32;
constexpr int RS_TILE = RS_THREADS * RS_ITEMS;  // 8192 elements per block
constexpr int RS_MAX_BINS = 256;

struct SortCtl {           // lives in the workspace
  unsigned long long R;    // true number of duplicated keys
  uint32_t overflow;       // 1 if R > capacity or R >= 2^32
  uint32_t pad;
};

// One stable radix pass on `bits` bits at `shift`.  kCount: write the per-block digit histogram to
// table[digit][block].  Otherwise: table holds the exclusive scan (digit-major) and the block
// scatters its elements, keeping their order within a digit.
template <bool kCount, bool kWriteKeys>
__global__ void __launch_bounds__(RS_THREADS) radix_pass_kernel(
    const uint32_t* __restrict__ keys_in, const uint32_t* __restrict__ vals_in, uint32_t* __restrict__ keys_out,
    uint32_t* __restrict__ vals_out, uint32_t n_static, const SortCtl* __restrict__ ctl, int shift, int bits,
    uint32_t* __restrict__ table, int nblocks) {
  __shared__ uint32_t cnt[RS_WARPS][RS_MAX_BINS];
  __shared__ uint32_t gbase[RS_MAX_BINS];
  const int bins = 1 << bits;
  uint32_t n = n_static;
  if (ctl) {
    if (ctl->overflow) n = 0;
    else n = (uint32_t)min((unsigned long long)n_static, ctl->R);
  }
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  for (int i = threadIdx.x; i < RS_WARPS * RS_MAX_BINS; i += RS_THREADS) (&cnt[0][0])[i] = 0;
  __syncthreads();
  const uint32_t base = blockIdx.x * (uint32_t)RS_TILE + warp * (32 * RS_ITEMS);
  const uint32_t mask = (uint32_t)bins - 1;
  uint32_t key[RS_ITEMS], rank[RS_ITEMS];
#pragma unroll
  for (int it = 0; it < RS_ITEMS; it++) {
    const uint32_t idx = base + it * 32 + lane;
    key[it] = idx < n ? keys_in[idx] : 0u;
  }
#pragma unroll
  for (int it = 0; it < RS_ITEMS; it++) {
    const uint32_t idx = base + it * 32 + lane;
    const bool valid = idx < n;
    const uint32_t d = valid ? ((key[it] >> shift) & mask) : (uint32_t)bins;  // invalid lanes match only each other
    const uint32_t peers = __match_any_sync(0xffffffffu, d);
    uint32_t before = 0;
    if (valid) before = cnt[warp][d];
    __syncwarp();
    if (valid && lane == __ffs(peers) - 1) cnt[warp][d] = before + __popc(peers);
    __syncwarp();
    rank[it] = before + __popc(peers & ((1u << lane) - 1u));
  }
  __syncthreads();
  if (threadIdx.x < bins) {
    uint32_t s = 0;
#pragma unroll
    for (int w = 0; w < RS_WARPS; w++) {
      const uint32_t c = cnt[w][threadIdx.x];
      cnt[w][threadIdx.x] = s;
      s += c;
    }
    if (kCount) table[(size_t)threadIdx.x * nblocks + blockIdx.x] = s;
    else gbase[threadIdx.x] = table[(size_t)threadIdx.x * nblocks + blockIdx.x];
  }
  if (kCount) return;
  __syncthreads();
#pragma unroll
  for (int it = 0; it < RS_ITEMS; it++) {
    const uint32_t idx = base + it * 32 + lane;
    if (idx < n) {
      const uint32_t d = (key[it] >> shift) & mask;
      const uint32_t dst = gbase[d] + cnt[warp][d] + rank[it];
      if (kWriteKeys) keys_out[dst] = key[it];
      vals_out[dst] = vals_in[idx];
    }
  }
}

// In-place exclusive scan of `total` uint32 values by one block (digit-major histogram table).
__global__ void __launch_bounds__(1024) table_scan_kernel(uint32_t* __restrict__ table, size_t total) {
  __shared__ uint32_t part[1024];
  const size_t chunk = (total + 1023) / 1024;
  const size_t b = (size_t)threadIdx.x * chunk, e = min(total, b + chunk);
  uint32_t s = 0;
  for (size_t i = b; i < e; i++) s += table[i];
  part[threadIdx.x] = s;
  __syncthreads();
  for (int o = 1; o < 1024; o <<= 1) {  // Hillis-Steele inclusive scan
    const uint32_t v = threadIdx.x >= o ? part[threadIdx.x - o] : 0;
    __syncthreads();
    part[threadIdx.x] += v;
    __syncthreads();
  }
  uint32_t run = part[threadIdx.x] - s;
  for (size_t i = b; i < e; i++) {
    const uint32_t v = table[i];
    table[i] = run;
    run += v;
  }
}

// Depth keys: fp32 bits of depth (positive floats order as unsigned ints); culled Gaussians last.
__global__ void depth_keys_kernel(int64_t N, const float* __restrict__ depths, const uint32_t* __restrict__ tiles_touched,
                                  uint32_t* __restrict__ keys, uint32_t* __restrict__ vals) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N) return;
  keys[i] = tiles_touched[i] ? __float_as_uint(depths[i]) : 0xffffffffu;
  vals[i] = (uint32_t)i;
}

__device__ __forceinline__ unsigned long long block_exclusive_scan_256(unsigned long long v, unsigned long long* total) {
  __shared__ unsigned long long wsum[8];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  unsigned long long inc = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const unsigned long long t = __shfl_up_sync(0xffffffffu, inc, o);
    if (lane >= o) inc += t;
  }
  if (lane == 31) wsum[warp] = inc;
  __syncthreads();
  unsigned long long woff = 0, tot = 0;
#pragma unroll
  for (int w = 0; w < 8; w++) {
    if (w < warp) woff += wsum[w];
    tot += wsum[w];
  }
  *total = tot;
  return woff + inc - v;
}

// Block sums of tiles_touched taken in depth order.
__global__ void __launch_bounds__(256) tt_block_sums_kernel(int64_t N, const uint32_t* __restrict__ order,
                                                            const uint32_t* __restrict__ tiles_touched,
                                                            unsigned long long* __restrict__ block_sums) {
  const int64_t k = (int64_t)blockIdx.x * 256 + threadIdx.x;
  const unsigned long long v = k < N ? tiles_touched[order[k]] : 0;
  unsigned long long tot;
  block_exclusive_scan_256(v, &tot);
  if (threadIdx.x == 0) block_sums[blockIdx.x] = tot;
}

// Exclusive scan of the block sums by one block; publishes R and the overflow flag.
__global__ void __launch_bounds__(1024) block_sums_scan_kernel(unsigned long long* __restrict__ block_sums, int nblk,
                                                               unsigned long long capacity, SortCtl* __restrict__ ctl,
                                                               int32_t* __restrict__ sat, int sat_n) {
  __shared__ unsigned long long part[1024];
  const int chunk = (nblk + 1023) / 1024;
  const int b = threadIdx.x * chunk, e = min(nblk, b + chunk);
  unsigned long long s = 0;
  for (int i = b; i < e; i++) s += block_sums[i];
  part[threadIdx.x] = s;
  __syncthreads();
  for (int o = 1; o < 1024; o <<= 1) {
    const unsigned long long v = threadIdx.x >= o ? part[threadIdx.x - o] : 0;
    __syncthreads();
    part[threadIdx.x] += v;
    __syncthreads();
  }
  unsigned long long run = part[threadIdx.x] - s;
  for (int i = b; i < e; i++) {
    const unsigned long long v = block_sums[i];
    block_sums[i] = run;
    run += v;
  }
  if (threadIdx.x == 1023) {
    ctl->R = part[1023];
    ctl->overflow = (part[1023] > capacity || part[1023] >= (1ull << 32)) ? 1u : 0u;
  }
  for (int i = threadIdx.x; i < sat_n; i += 1024) sat[i] = 0;
}

// Key duplication in depth order: entry k of the depth order writes its tile ids (row-major over its
// rectangle) at offset[k].  Rectangles with more than 16 tiles are written by the whole warp.
// Also scatters the four corners of the rectangle into the summed-area table.
__global__ void __launch_bounds__(256) duplicate_kernel(int64_t N, const uint32_t* __restrict__ order,
                                                        const uint32_t* __restrict__ tiles_touched,
                                                        const int4* __restrict__ rects,
                                                        const unsigned long long* __restrict__ block_offsets,
                                                        const SortCtl* __restrict__ ctl, int gw, int gh,
                                                        uint32_t* __restrict__ tile_keys, uint32_t* __restrict__ ids,
                                                        int32_t* __restrict__ sat) {
  if (ctl->overflow) return;
  const int64_t k = (int64_t)blockIdx.x * 256 + threadIdx.x;
  uint32_t id = 0, cnt = 0;
  int4 r = make_int4(0, 0, 0, 0);
  if (k < N) {
    id = order[k];
    cnt = tiles_touched[id];
    if (cnt) r = rects[id];
  }
  unsigned long long tot;
  const unsigned long long off64 = block_offsets[blockIdx.x] + block_exclusive_scan_256(cnt, &tot);
  const uint32_t off = (uint32_t)off64;
  if (cnt) {
    const int sw = gw + 1;
    atomicAdd(&sat[r.y * sw + r.x], 1);
    atomicAdd(&sat[r.y * sw + r.z], -1);
    atomicAdd(&sat[r.w * sw + r.x], -1);
    atomicAdd(&sat[r.w * sw + r.z], 1);
  }
  const int lane = threadIdx.x & 31;
  const bool big = cnt > 16;
  if (cnt && !big) {
    uint32_t o = off;
    for (int y = r.y; y < r.w; y++)
      for (int x = r.x; x < r.z; x++) {
        tile_keys[o] = (uint32_t)(y * gw + x);
        ids[o] = id;
        o++;
      }
  }
  uint32_t todo = __ballot_sync(0xffffffffu, big);
  while (todo) {
    const int src = __ffs(todo) - 1;
    todo &= todo - 1;
    const uint32_t bid = __shfl_sync(0xffffffffu, id, src), bcnt = __shfl_sync(0xffffffffu, cnt, src);
    const uint32_t boff = __shfl_sync(0xffffffffu, off, src);
    const int bx0 = __shfl_sync(0xffffffffu, r.x, src), by0 = __shfl_sync(0xffffffffu, r.y, src);
    const int bw = __shfl_sync(0xffffffffu, r.z, src) - bx0;
    for (uint32_t j = lane; j < bcnt; j += 32) {
      const int y = by0 + (int)(j / (uint32_t)bw), x = bx0 + (int)(j % (uint32_t)bw);
      tile_keys[boff + j] = (uint32_t)(y * gw + x);
      ids[boff + j] = bid;
    }
  }
}

// Tile ranges from the summed-area table: 2D prefix sum -> keys per tile -> exclusive scan.
__global__ void __launch_bounds__(1024) tile_ranges_kernel(int32_t* __restrict__ sat, int gw, int gh,
                                                           const SortCtl* __restrict__ ctl, uint32_t* __restrict__ tile_ranges) {
  __shared__ uint32_t part[1024];
  const int ntiles = gw * gh, sw = gw + 1;
  if (ctl->overflow) {
    for (int t = threadIdx.x; t < ntiles; t += 1024) { tile_ranges[2 * t] = 0; tile_ranges[2 * t + 1] = 0; }
    return;
  }
  for (int y = threadIdx.x; y < gh; y += 1024) {  // prefix along x
    int run = 0;
    for (int x = 0; x < gw; x++) { run += sat[y * sw + x]; sat[y * sw + x] = run; }
  }
  __syncthreads();
  for (int x = threadIdx.x; x < gw; x += 1024) {  // prefix along y: sat[y][x] = keys of tile (x, y)
    int run = 0;
    for (int y = 0; y < gh; y++) { run += sat[y * sw + x]; sat[y * sw + x] = run; }
  }
  __syncthreads();
  const int chunk = (ntiles + 1023) / 1024;
  const int b = threadIdx.x * chunk, e = min(ntiles, b + chunk);
  uint32_t s = 0;
  for (int t = b; t < e; t++) s += (uint32_t)sat[(t / gw) * sw + (t % gw)];
  part[threadIdx.x] = s;
  __syncthreads();
  for (int o = 1; o < 1024; o <<= 1) {
    const uint32_t v = threadIdx.x >= o ? part[threadIdx.x - o] : 0;
    __syncthreads();
    part[threadIdx.x] += v;
    __syncthreads();
  }
  uint32_t run = part[threadIdx.x] - s;
  for (int t = b; t < e; t++) {
    const uint32_t c = (uint32_t)sat[(t / gw) * sw + (t % gw)];
    tile_ranges[2 * t] = run;
    run += c;
    tile_ranges[2 * t + 1] = run;
  }
}

struct Layout {
  size_t ctl, keysA, valsA, keysB, valsB, block_sums, table, sat, tkA, tiA, tkB, tiB, total;
  int nblkN_scan, nblkN_sort, nblkR_sort;
  int tile_bits, tile_passes, bits_per_pass;
};

inline size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }

Layout make_layout(int64_t N, int gw, int gh, uint64_t Rcap) {
  Layout L;
  const size_t n = (size_t)N, r = (size_t)Rcap;
  const int ntiles = gw * gh;
  L.tile_bits = 1;
  while ((1ll << L.tile_bits) < ntiles) L.tile_bits++;
  L.tile_passes = (L.tile_bits + 7) / 8;
  L.bits_per_pass = (L.tile_bits + L.tile_passes - 1) / L.tile_passes;
  L.nblkN_scan = (int)((n + 255) / 256);
  L.nblkN_sort = (int)((n + RS_TILE - 1) / RS_TILE);
  L.nblkR_sort = (int)((r + RS_TILE - 1) / RS_TILE);
  size_t o = 0;
  L.ctl = o; o = align256(o + sizeof(SortCtl));
  L.keysA = o; o = align256(o + 4 * n);
  L.valsA = o; o = align256(o + 4 * n);
  L.keysB = o; o = align256(o + 4 * n);
  L.valsB = o; o = align256(o + 4 * n);
  L.block_sums = o; o = align256(o + 8 * (size_t)(L.nblkN_scan + 1));
  const size_t tab = (size_t)RS_MAX_BINS * (size_t)(L.nblkN_sort > L.nblkR_sort ? L.nblkN_sort : L.nblkR_sort);
  L.table = o; o = align256(o + 4 * (tab + 1));
  L.sat = o; o = align256(o + 4 * (size_t)(gw + 1) * (gh + 1));
  L.tkA = o; o = align256(o + 4 * r);
  L.tiA = o; o = align256(o + 4 * r);
  L.tkB = o; o = align256(o + (L.tile_passes > 1 ? 4 * r : 0));
  L.tiB = o; o = align256(o + (L.tile_passes > 1 ? 4 * r : 0));
  L.total = o;
  return L;
}

}  // namespace

extern "C" size_t mg_workspace_bytes(int64_t N, int32_t width, int32_t height, uint64_t R_capacity) {
  if (N < 0 || width <= 0 || height <= 0 || R_capacity >= (1ull << 32)) return 0;
  const int gw = (width + MG_TILE - 1) / MG_TILE, gh = (height + MG_TILE - 1) / MG_TILE;
  return make_layout(N, gw, gh, R_capacity).total;
}

extern "C" int mg_bin_sort(const mg_camera* cam, int64_t N, const float* depths, const int32_t* rects,
                           const uint32_t* tiles_touched, uint64_t R_capacity, void* workspace, size_t workspace_bytes,
                           uint32_t* sorted_ids, uint32_t* tile_ranges, uint64_t* R_out_host, void* stream) {
  if (int rc = mg_check_camera(cam)) return rc;
  MG_REQUIRE(N >= 0 && N < (int64_t)1 << 31, "N must be in [0, 2^31)");
  MG_REQUIRE(R_capacity < (1ull << 32), "R_capacity must be < 2^32");
  MG_REQUIRE(tile_ranges != nullptr, "tile_ranges is null");
  MG_REQUIRE(workspace != nullptr && ((uintptr_t)workspace & 255) == 0, "workspace must be non-null and 256-byte aligned");
  MG_REQUIRE(N == 0 || (depths && rects && tiles_touched), "null input array");
  MG_REQUIRE(R_capacity == 0 || sorted_ids != nullptr, "sorted_ids is null");
  const int gw = mg_grid_w(cam), gh = mg_grid_h(cam);
  const Layout L = make_layout(N, gw, gh, R_capacity);
  if (workspace_bytes < L.total) {
    mg_set_error("workspace too small: %zu bytes given, %zu needed", workspace_bytes, L.total);
    return MG_ERR_CAPACITY;
  }
  cudaStream_t st = (cudaStream_t)stream;
  char* ws = (char*)workspace;
  SortCtl* ctl = (SortCtl*)(ws + L.ctl);
  uint32_t *keysA = (uint32_t*)(ws + L.keysA), *valsA = (uint32_t*)(ws + L.valsA);
  uint32_t *keysB = (uint32_t*)(ws + L.keysB), *valsB = (uint32_t*)(ws + L.valsB);
  unsigned long long* block_sums = (unsigned long long*)(ws + L.block_sums);
  uint32_t* table = (uint32_t*)(ws + L.table);
  int32_t* sat = (int32_t*)(ws + L.sat);
  uint32_t *tkA = (uint32_t*)(ws + L.tkA), *tiA = (uint32_t*)(ws + L.tiA);
  uint32_t *tkB = (uint32_t*)(ws + L.tkB), *tiB = (uint32_t*)(ws + L.tiB);
  const int sat_n = (gw + 1) * (gh + 1);

  // (1) depth order of the N Gaussians: stable LSD radix sort of the fp32 depth bits, 4 x 8 bits
  if (N > 0) {
    depth_keys_kernel<<<(unsigned)((N + 255) / 256), 256, 0, st>>>(N, depths, tiles_touched, keysA, valsA);
    MG_CHECK_LAUNCH();
    uint32_t *ki = keysA, *vi = valsA, *ko = keysB, *vo = valsB;
    for (int pass = 0; pass < 4; pass++) {
      radix_pass_kernel<true, false><<<L.nblkN_sort, RS_THREADS, 0, st>>>(ki, vi, ko, vo, (uint32_t)N, nullptr, 8 * pass, 8, table, L.nblkN_sort);
      table_scan_kernel<<<1, 1024, 0, st>>>(table, (size_t)256 * L.nblkN_sort);
      radix_pass_kernel<false, true><<<L.nblkN_sort, RS_THREADS, 0, st>>>(ki, vi, ko, vo, (uint32_t)N, nullptr, 8 * pass, 8, table, L.nblkN_sort);
      MG_CHECK_LAUNCH();
      uint32_t* t = ki; ki = ko; ko = t;
      t = vi; vi = vo; vo = t;
    }
    // after 4 passes the result is back in (keysA, valsA)
    tt_block_sums_kernel<<<L.nblkN_scan, 256, 0, st>>>(N, valsA, tiles_touched, block_sums);
    MG_CHECK_LAUNCH();
  }
  // (2) offsets of each Gaussian's run of keys; R and the overflow flag; clears the summed-area table
  block_sums_scan_kernel<<<1, 1024, 0, st>>>(block_sums, N > 0 ? L.nblkN_scan : 0, R_capacity, ctl, sat, sat_n);
  MG_CHECK_LAUNCH();
  if (N > 0) {
    // (3) duplication in depth order
    uint32_t* first_ids = (L.tile_passes == 0) ? sorted_ids : tiA;
    duplicate_kernel<<<L.nblkN_scan, 256, 0, st>>>(N, valsA, tiles_touched, (const int4*)rects, block_sums, ctl, gw, gh, tkA, first_ids, sat);
    MG_CHECK_LAUNCH();
    // (4) stable passes over the tile bits; the last one writes only the ids, to sorted_ids
    if (R_capacity > 0) {
      uint32_t *ki = tkA, *vi = tiA, *ko = tkB, *vo = tiB;
      for (int pass = 0; pass < L.tile_passes; pass++) {
        const bool last = pass == L.tile_passes - 1;
        const int shift = pass * L.bits_per_pass;
        radix_pass_kernel<true, false><<<L.nblkR_sort, RS_THREADS, 0, st>>>(ki, vi, ko, vo, (uint32_t)R_capacity, ctl, shift, L.bits_per_pass, table, L.nblkR_sort);
        table_scan_kernel<<<1, 1024, 0, st>>>(table, ((size_t)1 << L.bits_per_pass) * L.nblkR_sort);
        if (last)
          radix_pass_kernel<false, false><<<L.nblkR_sort, RS_THREADS, 0, st>>>(ki, vi, nullptr, sorted_ids, (uint32_t)R_capacity, ctl, shift, L.bits_per_pass, table, L.nblkR_sort);
        else
          radix_pass_kernel<false, true><<<L.nblkR_sort, RS_THREADS, 0, st>>>(ki, vi, ko, vo, (uint32_t)R_capacity, ctl, shift, L.bits_per_pass, table, L.nblkR_sort);
        MG_CHECK_LAUNCH();
        uint32_t* t = ki; ki = ko; ko = t;
        t = vi; vi = vo; vo = t;
      }
    }
  }
  // (5) tile ranges
  tile_ranges_kernel<<<1, 1024, 0, st>>>(sat, gw, gh, ctl, tile_ranges);
  MG_CHECK_LAUNCH();
  if (R_out_host) MG_CHECK_CUDA(cudaMemcpyAsync(R_out_host, &ctl->R, sizeof(uint64_t), cudaMemcpyDeviceToHost, st));
  return MG_OK;
}
