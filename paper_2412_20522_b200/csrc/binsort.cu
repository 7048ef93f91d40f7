// binsort.cu -- mg_bin_sort: key duplication, (tile, depth) sort, tile ranges.
// Steps a4-a6 of the hot path (PAPER.md:66 "depth order", :74 16x16 tiles; O9).
//
// The result is DEFINED as the ascending order of the 64-bit keys (tile_id << 32 | depth bits), ties
// by Gaussian index, tile_id = ty * gw + tx.  It is produced without ever materialising those keys:
//
//  S1  depth order of the VISIBLE Gaussians: stable LSD radix sort of the fp32 depth bits (4 x 8 bits).
//      All duplicates of a Gaussian share its depth, so the depth digits are sorted BEFORE the
//      duplication (nvis keys instead of R).  The first pass reads depths and tiles_touched themselves and
//      neither ranks nor writes a culled Gaussian, so the other three passes move the visible ones only.
//  S2  row expansion: Gaussian k of the depth order covers tile rows [y0, y1); it emits one record
//      (id, x0, x1) into the list of each of those rows, lists kept in depth order.  All duplicates
//      of a Gaussian within a tile row share (depth, ty), so the row digit is "sorted" before the
//      expansion in x (sum(y1 - y0) records instead of R).
//  S3  column expansion: within a row, record j covers tile columns [x0, x1); it emits its id into
//      the list of each of those tiles, lists kept in record order.  The concatenation of the tile
//      lists over (ty, tx) ascending is sorted_ids; the list boundaries are tile_ranges.
//
// S2 and S3 are the same primitive, a STABLE INTERVAL EXPANSION: items in sequence order, each with
// an interval of bins, are appended to every bin of their interval, order preserved.  A warp takes
// a chunk of 128 consecutive items, 32 at a time.  Counting: a difference array per chunk in shared
// memory (two atomics per item), scanned over the bins at the end.  Per chunk and bin the counts go
// to a table, an exclusive scan of the table (bin-major, chunk-minor) gives every (bin, chunk) its
// write position, and a second sweep emits: lane k turns its interval into a row of a 32 x 32-bin bit
// matrix, a 5-stage shuffle butterfly transposes it, and lane c then holds the set of items that cover
// bin c, in item order, and walks the set bits.  (A lanes-as-keys variant -- binary search over the
// scanned widths, then ranking by match -- was measured 1.5x slower: longer dependent chains.)
//
// Bytes moved per duplicated key: ~4 B written + ~16 B of records and tables (mostly L2 hits),
// against ~150 B for six 64-bit key-value radix passes over R keys.
#include <atomic>

#include "mg_common.cuh"

namespace {

// ---------------------------------------------------------------- S1: radix sort of the N depth keys
#ifndef RS_THREADS_
#define RS_THREADS_ 512
#endif
#ifndef RS_ITEMS_
#define RS_ITEMS_ 8
#endif
constexpr int RS_THREADS = RS_THREADS_;
constexpr int RS_ITEMS = RS_ITEMS_;
constexpr int RS_WARPS = RS_THREADS / 32;
constexpr int RS_TILE = RS_THREADS * RS_ITEMS;  // 4096 elements per block: 41 KB of shared memory, 5 blocks per SM
constexpr int RS_BINS = 256;

#ifndef XP_CHUNK_
#define XP_CHUNK_ 128
#endif
constexpr int XP_CHUNK = XP_CHUNK_;   // items per warp in the expansion sweeps
constexpr int XP_GROUPS = XP_CHUNK / 32;
constexpr int XP_MAX_WARPS = 8; // warps per block in the expansion sweeps
constexpr int SCAN_THREADS = 1024;
constexpr int SCAN_ITEMS = 4;
constexpr int SCAN_BLK = SCAN_THREADS * SCAN_ITEMS;

constexpr int TO_CLASSES = 257;  // list-length classes of the scheduling hint tile_order

// class(0) = 0, class(n) = 1 + 8 floor(log2 n) + the next 3 bits of n: monotone in n, integer-only.
__device__ __forceinline__ uint32_t length_class(uint32_t n) {
  if (n == 0) return 0u;
  const int msb = 31 - __clz(n);
  const uint32_t frac = msb >= 3 ? (n >> (msb - 3)) & 7u : (n << (3 - msb)) & 7u;
  return 1u + 8u * (uint32_t)msb + frac;
}

// Lanes with the same `nbits`-bit value among the lanes of `vmask` (the caller's own lane included), built
// from one ballot per bit.  On sm_100a this is several times faster than match.any, whose cost made it the
// bottleneck of every ranking loop here.
__device__ __forceinline__ uint32_t peers_by_ballot(uint32_t v, int nbits, uint32_t vmask) {
  uint32_t peers = vmask;
  for (int b = 0; b < nbits; b++) {
    const bool bit = (v >> b) & 1u;
    const uint32_t set = __ballot_sync(0xffffffffu, bit);
    peers &= bit ? set : ~set;
  }
  return peers;
}

struct SortCtl {            // lives in the workspace; zeroed at the start of every call
  unsigned long long R;     // true number of duplicated keys = sum of tiles_touched
  uint32_t nvis;            // Gaussians with tiles_touched > 0
  uint32_t overflow;        // 1 if R > capacity or R >= 2^32; 2 if a look-back gave up (nothing is emitted either way)
  uint32_t n_chunks_c;      // chunks of the column expansion (sum over rows of ceil(records / XP_CHUNK))
  uint32_t n_table_c;       // gw * n_chunks_c
  uint32_t pad[2];
  uint32_t ticket[4];       // next logical tile of each radix pass (tiles are taken in ticket order)
  uint32_t pad2[4];
  uint32_t ghist[4][RS_BINS];  // digit histograms of the depth keys, all four passes; then exclusive bases
  uint32_t class_count[TO_CLASSES];   // tiles per list-length class (tile_order)
  uint32_t class_cursor[TO_CLASSES];  // tiles of the class already placed
};

// Shared memory of a radix pass.  The block ranks its keys (per-warp digit counters, warps in order), moves
// keys and values into digit order in shared memory, and writes them out from there, so that consecutive
// threads write consecutive addresses of a digit's run.
struct RadixSmem {
  uint32_t cnt[RS_WARPS][RS_BINS];  // per-warp digit counts -> exclusive prefix over warps
  uint32_t lbase[RS_BINS];          // first local position of a digit
  uint32_t gdelta[RS_BINS];         // global position of a digit's first key minus its local position
  uint32_t keys[RS_TILE];
  uint32_t vals[RS_TILE];
};

__device__ __forceinline__ void st_relaxed_u64(unsigned long long* p, unsigned long long v) {
  asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}
__device__ __forceinline__ unsigned long long ld_relaxed_u64(const unsigned long long* p) {
  unsigned long long v;
  asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
  return v;
}

// ---- programmatic dependent launch (sm_90+).  mg_bin_sort is a chain of 17 short kernels, eight of them 5-16 us
// long, each of which depends on all of its predecessor: between two such kernels the GPU idles for the launch latency
// and the drain of the last blocks.  Launched with cudaLaunchAttributeProgrammaticStreamSerialization, a kernel's blocks
// may become resident while its predecessor is still running; every kernel of this file therefore begins with
// pdl_prologue(): griddepcontrol.wait blocks until the predecessor grid has COMPLETED and its writes are visible (so
// nothing of the dependency is given up -- not a load, not a store happens before it, which also covers buffers the
// predecessor still reads), then griddepcontrol.launch_dependents lets the successor's blocks be scheduled as soon as
// every block of this grid has started.  What is gained is the launch latency and the tail, nothing else.  Both
// instructions are no-ops in a kernel launched without the attribute (the first kernel after a memset, MG_NO_PDL).
__device__ __forceinline__ void pdl_prologue() {
  asm volatile("griddepcontrol.wait;" ::: "memory");
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
}

constexpr unsigned long long LB_AGGREGATE = 1ull << 32;  // status word = flag << 32 | count
constexpr unsigned long long LB_INCLUSIVE = 2ull << 32;
constexpr int LB_SPIN_LIMIT = 1 << 26;                   // polls of one status word before a look-back gives up
#ifdef MG_TESTING  // the test build only (libmg_testing.so): the shipped library has neither the hook nor its state
std::atomic<int> g_spin_limit{LB_SPIN_LIMIT};             // mg_debug_set_lookback_spin_limit (failure injection in tests)
#endif

// One radix pass = ONE kernel (single-pass chained scan with decoupled look-back): a block takes the next
// logical tile by ticket, ranks its 4096 keys, publishes its per-digit counts, and obtains its per-digit
// offsets by summing the counts its predecessors have published (an "aggregate" if that tile has only
// counted, an "inclusive" total -- which ends the walk -- once it has finished its own look-back).  Tiles
// are taken in ticket order, so a block only ever waits for blocks that started before it.  The digit
// bases of the whole array come from the histograms depth_hist_kernel took.
// kFirst (pass 0): keys_in = the fp32 depths of ALL n_all Gaussians, vals_in = their tiles_touched.  A Gaussian with
// tiles_touched == 0 is neither ranked nor written (it is treated like an index past the end), its value is its index,
// and the tile writes as many keys as it has visible Gaussians.  Tiles, tickets and the stable order are unchanged, so
// the pass is at once the first digit pass and the compaction.  The other passes sort ctl->nvis keys; their grid is
// sized for n_all and the surplus blocks leave at once.
template <bool kFirst>
__global__ void __launch_bounds__(RS_THREADS) radix_onesweep_kernel(
    const uint32_t* __restrict__ keys_in, const uint32_t* __restrict__ vals_in, uint32_t* __restrict__ keys_out,
    uint32_t* __restrict__ vals_out, uint32_t n_all, int pass, SortCtl* __restrict__ ctl,
    unsigned long long* __restrict__ status, int spin_limit) {
  pdl_prologue();
  extern __shared__ __align__(16) unsigned char rs_smem_raw[];
  RadixSmem& sm = *reinterpret_cast<RadixSmem*>(rs_smem_raw);
  __shared__ uint32_t s_tile, s_nvalid;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int shift = 8 * pass;
  const uint32_t n = kFirst ? n_all : ctl->nvis;
  // exactly ceil(n / RS_TILE) blocks stay, and they take exactly the tickets below that number
  if ((uint64_t)blockIdx.x * RS_TILE >= n) return;
  if (threadIdx.x == 0) s_tile = atomicAdd(&ctl->ticket[pass], 1u);
  for (int i = threadIdx.x; i < RS_WARPS * RS_BINS; i += RS_THREADS) (&sm.cnt[0][0])[i] = 0;
  __syncthreads();
  const uint32_t tile = s_tile;
  const uint32_t base = tile * (uint32_t)RS_TILE + warp * (32 * RS_ITEMS);
  uint32_t key[RS_ITEMS], val[RS_ITEMS], rank[RS_ITEMS];
  uint32_t vbits = 0;  // bit it: this thread's item it takes part in the sort
#pragma unroll
  for (int it = 0; it < RS_ITEMS; it++) {
    const uint32_t idx = base + it * 32 + lane;
    bool v = idx < n;
    if (kFirst) {
      v = v && vals_in[idx] != 0u;  // tiles_touched: culled Gaussians do not take part
      val[it] = idx;                // the value is the Gaussian's index
    } else {
      val[it] = v ? vals_in[idx] : 0u;
    }
    key[it] = v ? keys_in[idx] : 0u;
    vbits |= (v ? 1u : 0u) << it;
  }
#pragma unroll
  for (int it = 0; it < RS_ITEMS; it++) {
    const bool valid = (vbits >> it) & 1u;
    const uint32_t d = (key[it] >> shift) & 255u;
    const uint32_t peers = peers_by_ballot(d, 8, __ballot_sync(0xffffffffu, valid));
    uint32_t before = 0;
    if (valid) before = sm.cnt[warp][d];
    __syncwarp();
    if (valid && lane == __ffs(peers) - 1) sm.cnt[warp][d] = before + __popc(peers);
    __syncwarp();
    rank[it] = before + __popc(peers & ((1u << lane) - 1u));
  }
  __syncthreads();
  // exclusive prefix over warps per digit; the digit totals are published at once (aggregate)
  uint32_t total = 0;
  unsigned long long* my_status = status + (size_t)tile * RS_BINS + threadIdx.x;
  if (threadIdx.x < RS_BINS) {
#pragma unroll
    for (int w = 0; w < RS_WARPS; w++) {
      const uint32_t c = sm.cnt[w][threadIdx.x];
      sm.cnt[w][threadIdx.x] = total;
      total += c;
    }
    st_relaxed_u64(my_status, LB_AGGREGATE | total);
  }
  {
    // exclusive scan of the totals over the 256 digits -> first local position of a digit
    uint32_t inc = total;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
      if (lane >= o) inc += t;
    }
    if (threadIdx.x < RS_BINS && lane == 31) sm.gdelta[warp] = inc;  // scratch: sums of warps 0..7
    __syncthreads();
    if (threadIdx.x < RS_BINS) {
      uint32_t woff = 0;
#pragma unroll
      for (int w = 0; w < RS_BINS / 32; w++)
        if (w < warp) woff += sm.gdelta[w];
      sm.lbase[threadIdx.x] = woff + inc - total;
      if (threadIdx.x == RS_BINS - 1) s_nvalid = woff + inc;  // keys of this tile that take part
    }
    __syncthreads();
  }
  if (threadIdx.x < RS_BINS) {
    // decoupled look-back over the tiles before this one, one digit per thread
    uint32_t prefix = 0;
    for (int t = (int)tile - 1; t >= 0; t--) {
      const unsigned long long* ps = status + (size_t)t * RS_BINS + threadIdx.x;
      unsigned long long w = ld_relaxed_u64(ps);
      int spins = 0;
      while ((w >> 32) == 0 && ++spins < spin_limit) w = ld_relaxed_u64(ps);
      // A predecessor that never publishes cannot happen (tiles are taken in ticket order, so it is resident and
      // running); if it does, the call fails loudly: nothing is emitted and R_out_host reads UINT64_MAX.
      if ((w >> 32) == 0 || spin_limit == 0) { ctl->overflow = 2u; break; }
      prefix += (uint32_t)w;
      if ((w & LB_INCLUSIVE) != 0) break;
    }
    st_relaxed_u64(my_status, LB_INCLUSIVE | (unsigned long long)(prefix + total));
    sm.gdelta[threadIdx.x] = ctl->ghist[pass][threadIdx.x] + prefix - sm.lbase[threadIdx.x];
  }
  // into digit order in shared memory
#pragma unroll
  for (int it = 0; it < RS_ITEMS; it++) {
    if ((vbits >> it) & 1u) {
      const uint32_t d = (key[it] >> shift) & 255u;
      const uint32_t lpos = sm.lbase[d] + sm.cnt[warp][d] + rank[it];
      sm.keys[lpos] = key[it];
      sm.vals[lpos] = val[it];
    }
  }
  __syncthreads();
  const uint32_t nblk = s_nvalid;
#pragma unroll
  for (int it = 0; it < RS_ITEMS; it++) {
    const uint32_t j = it * RS_THREADS + threadIdx.x;
    if (j < nblk) {
      const uint32_t k = sm.keys[j];
      const uint32_t dst = sm.gdelta[(k >> shift) & 255u] + j;
      keys_out[dst] = k;
      vals_out[dst] = sm.vals[j];
    }
  }
}

// The sort key of a Gaussian is the fp32 bit pattern of its depth (positive floats order as unsigned ints); only
// VISIBLE Gaussians (tiles_touched > 0) are sorted.  This kernel takes, in one read of depths and tiles_touched, the
// digit histograms of all four radix passes over the visible keys (they do not depend on the order of the keys),
// R = sum of tiles_touched and the number of visible Gaussians.  It writes no keys: the first radix pass reads the
// depths itself.
__global__ void __launch_bounds__(256) depth_hist_kernel(int64_t N, const float* __restrict__ depths,
                                                         const uint32_t* __restrict__ tiles_touched,
                                                         SortCtl* __restrict__ ctl) {
  pdl_prologue();
  __shared__ unsigned long long s_sum[8];
  __shared__ uint32_t s_vis[8];
  __shared__ uint32_t hist[4][RS_BINS];
  for (int j = threadIdx.x; j < 4 * RS_BINS; j += 256) (&hist[0][0])[j] = 0;
  __syncthreads();
  unsigned long long sum = 0;
  uint32_t vis = 0;
  for (int64_t i = (int64_t)blockIdx.x * 256 + threadIdx.x; i < N; i += (int64_t)gridDim.x * 256) {
    const uint32_t tt = tiles_touched[i];
    sum += tt;
    vis += tt != 0;
    if (tt) {
      const uint32_t key = __float_as_uint(depths[i]);
#pragma unroll
      for (int p = 0; p < 4; p++) atomicAdd(&hist[p][(key >> (8 * p)) & 255u], 1u);
    }
  }
#pragma unroll
  for (int o = 16; o >= 1; o >>= 1) {
    sum += __shfl_xor_sync(0xffffffffu, sum, o);
    vis += __shfl_xor_sync(0xffffffffu, vis, o);
  }
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  if (lane == 0) { s_sum[warp] = sum; s_vis[warp] = vis; }
  __syncthreads();
  if (threadIdx.x == 0) {
    unsigned long long t = 0;
    uint32_t v = 0;
#pragma unroll
    for (int w = 0; w < 8; w++) { t += s_sum[w]; v += s_vis[w]; }
    if (t) atomicAdd(&ctl->R, t);
    if (v) atomicAdd(&ctl->nvis, v);
  }
  for (int j = threadIdx.x; j < 4 * RS_BINS; j += 256) {
    const uint32_t c = (&hist[0][0])[j];
    if (c) atomicAdd(&ctl->ghist[0][0] + j, c);
  }
}

// Overflow flag; digit histograms -> exclusive digit bases (one block of 256 threads).
__global__ void __launch_bounds__(RS_BINS) ctl_finalize_kernel(SortCtl* __restrict__ ctl, unsigned long long capacity) {
  pdl_prologue();
  __shared__ uint32_t h[4][RS_BINS];
  if (threadIdx.x == 0) ctl->overflow = (ctl->R > capacity || ctl->R >= (1ull << 32)) ? 1u : 0u;
  for (int p = 0; p < 4; p++) h[p][threadIdx.x] = ctl->ghist[p][threadIdx.x];
  __syncthreads();
  for (int p = 0; p < 4; p++) {
    uint32_t run = 0;
    for (int d = 0; d < (int)threadIdx.x; d++) run += h[p][d];
    ctl->ghist[p][threadIdx.x] = run;
  }
}

// ---------------------------------------------------------------- exclusive scan of a uint32 table
// Two launches: per-block sums, then each block adds the sums of the blocks before it and scans its
// own part in place.  n comes from device memory when n_dev != nullptr (else n_static).  The grand
// total is written to table[n].
__device__ __forceinline__ uint32_t scan_n(uint32_t n_static, const uint32_t* n_dev) { return n_dev ? *n_dev : n_static; }

__device__ __forceinline__ uint32_t block_reduce_1024(uint32_t v, uint32_t* sh) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  v = __reduce_add_sync(0xffffffffu, v);
  __syncthreads();  // sh may still be read from a previous use
  if (lane == 0) sh[warp] = v;
  __syncthreads();
  uint32_t t = sh[lane];
  t = __reduce_add_sync(0xffffffffu, t);
  return t;
}

__global__ void __launch_bounds__(SCAN_THREADS) scan_sums_kernel(const uint32_t* __restrict__ table, uint32_t n_static,
                                                                 const uint32_t* __restrict__ n_dev,
                                                                 uint32_t* __restrict__ sums) {
  pdl_prologue();
  __shared__ uint32_t sh[32];
  const uint32_t n = scan_n(n_static, n_dev);
  const uint32_t b0 = blockIdx.x * (uint32_t)SCAN_BLK;
  if (b0 >= n) return;
  uint32_t s = 0;
#pragma unroll
  for (int i = 0; i < SCAN_ITEMS; i++) {
    const uint32_t idx = b0 + i * SCAN_THREADS + threadIdx.x;
    if (idx < n) s += table[idx];
  }
  s = block_reduce_1024(s, sh);
  if (threadIdx.x == 0) sums[blockIdx.x] = s;
}

__global__ void __launch_bounds__(SCAN_THREADS) scan_apply_kernel(uint32_t* __restrict__ table, uint32_t n_static,
                                                                  const uint32_t* __restrict__ n_dev,
                                                                  const uint32_t* __restrict__ sums) {
  pdl_prologue();
  __shared__ uint32_t sh[32];
  __shared__ uint32_t wsum[32];
  const uint32_t n = scan_n(n_static, n_dev);
  const uint32_t b0 = blockIdx.x * (uint32_t)SCAN_BLK;
  if (n == 0) {
    if (blockIdx.x == 0 && threadIdx.x == 0) table[0] = 0;
    return;
  }
  if (b0 >= n) return;
  uint32_t pre = 0;
  for (uint32_t j = threadIdx.x; j < blockIdx.x; j += SCAN_THREADS) pre += sums[j];
  pre = block_reduce_1024(pre, sh);
  // each thread owns SCAN_ITEMS consecutive elements
  const uint32_t t0 = b0 + threadIdx.x * SCAN_ITEMS;
  uint32_t v[SCAN_ITEMS], s = 0;
#pragma unroll
  for (int i = 0; i < SCAN_ITEMS; i++) {
    v[i] = (t0 + i < n) ? table[t0 + i] : 0u;
    s += v[i];
  }
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  uint32_t inc = s;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
    if (lane >= o) inc += t;
  }
  if (lane == 31) wsum[warp] = inc;
  __syncthreads();
  uint32_t woff = 0, tot = 0;
  {
    const uint32_t w = wsum[lane];
    uint32_t winc = w;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const uint32_t t = __shfl_up_sync(0xffffffffu, winc, o);
      if (lane >= o) winc += t;
    }
    woff = __shfl_sync(0xffffffffu, winc - w, warp);
    tot = __shfl_sync(0xffffffffu, winc, 31);
  }
  uint32_t run = pre + woff + inc - s;
#pragma unroll
  for (int i = 0; i < SCAN_ITEMS; i++) {
    if (t0 + i < n) table[t0 + i] = run;
    run += v[i];
  }
  if (b0 + SCAN_BLK >= n && threadIdx.x == 0) table[n] = pre + tot;
}

// ---------------------------------------------------------------- stable interval expansion
// Counting sweep, per warp and group of 32 items: a difference array in shared memory (+1 at lo, -1 at hi,
// two atomics per ITEM, not per key); xp_counts_to_table turns it into per-bin counts at the end of the chunk.
__device__ __forceinline__ void xp_count_group(int lo, int hi, uint32_t* cnt) {
  if (hi > lo) {
    atomicAdd(&cnt[lo], 1u);
    atomicSub(&cnt[hi], 1u);  // cnt has bins + 1 entries
  }
}

// Inclusive scan of the difference array over the bins -> counts; written to table[b * stride] (b < bins).
__device__ __forceinline__ void xp_counts_to_table(const uint32_t* cnt, int bins, int lane, uint32_t* table, size_t stride) {
  uint32_t carry = 0;
  for (int b0 = 0; b0 < bins; b0 += 32) {
    const int b = b0 + lane;
    uint32_t v = b < bins ? cnt[b] : 0u;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const uint32_t t = __shfl_up_sync(0xffffffffu, v, o);
      if (lane >= o) v += t;
    }
    v += carry;
    if (b < bins) table[(size_t)b * stride] = v;
    carry = __shfl_sync(0xffffffffu, v, 31);
  }
}

// Bits [lo, hi) of the 32-bin word w.
__device__ __forceinline__ uint32_t interval_bits(int lo, int hi, int w) {
  const int l = max(lo - 32 * w, 0), h = min(hi - 32 * w, 32);
  if (h <= l) return 0u;
  const uint32_t upto_h = h >= 32 ? 0xffffffffu : ((1u << h) - 1u);
  return upto_h & ~((1u << l) - 1u);
}

// 32 x 32 bit-matrix transpose across a warp: in, lane k holds row k (bit c = column c); out, lane c
// holds column c (bit k = row k).
__device__ __forceinline__ uint32_t transpose32(uint32_t x, int lane) {
#pragma unroll
  for (int j = 16; j >= 1; j >>= 1) {
    const uint32_t m = j == 16 ? 0x0000ffffu : j == 8 ? 0x00ff00ffu : j == 4 ? 0x0f0f0f0fu : j == 2 ? 0x33333333u : 0x55555555u;
    const uint32_t y = __shfl_xor_sync(0xffffffffu, x, j);
    if (lane & j) x = ((y >> j) & m) | (x & ~m);
    else x = (x & m) | ((y << j) & ~m);
  }
  return x;
}

// Word range [wlo, whi] touched by the valid intervals of a warp's 32 items (whi < wlo if none).
__device__ __forceinline__ void word_range(int lo, int hi, int* wlo, int* whi) {
  const bool any = hi > lo;
  *wlo = (int)__reduce_min_sync(0xffffffffu, any ? (uint32_t)(lo >> 5) : 0x7fffffffu);
  *whi = (int)__reduce_max_sync(0xffffffffu, any ? (hi - 1) >> 5 : -1);
}

// Emitting sweep, per warp and group of 32 items (lane k holds item k: interval [lo, hi), payload p0 and, if
// kWords == 2, p1): lane k turns its interval into a row of a 32 x 32-bin bit matrix per 32-bin word, a
// 5-stage shuffle butterfly transposes it, and lane c then holds the set of items that cover bin c, in
// item order; it walks the set bits and appends the payloads at the bin's write cursor cnt[bin].
template <int kWords>
__device__ __forceinline__ void xp_emit_group(int lo, int hi, uint32_t p0, uint32_t p1, uint32_t* cnt, int lane,
                                              uint32_t* __restrict__ out) {
  int wlo, whi;
  word_range(lo, hi, &wlo, &whi);
  for (int w = wlo; w <= whi; w++) {
    uint32_t col = transpose32(interval_bits(lo, hi, w), lane);
    const int bin = 32 * w + lane;
    const bool mine = col != 0;  // implies bin < bins
    uint32_t p = mine ? cnt[bin] : 0u;
    while (__any_sync(0xffffffffu, col != 0)) {
      const int src = col ? __ffs(col) - 1 : 0;
      const uint32_t v0 = __shfl_sync(0xffffffffu, p0, src);
      uint32_t v1 = 0;
      if (kWords == 2) v1 = __shfl_sync(0xffffffffu, p1, src);
      if (col) {
        if (kWords == 2) reinterpret_cast<uint2*>(out)[p++] = make_uint2(v0, v1);
        else out[p++] = v0;
        col &= col - 1;
      }
    }
    if (mine) cnt[bin] = p;
  }
}

// S2: row expansion.  Item k of the depth order (k < nvis) covers rows [y0, y1).
// kCount: table_r[row * n_chunks + chunk] = number of records of this chunk in that row; also stores the
// packed rectangle in depth order for the second sweep.  Otherwise table_r is scanned and the records
// (id, x0 | x1 << 16) are written to row_rec at their positions.
template <bool kCount>
__global__ void __launch_bounds__(32 * XP_MAX_WARPS) row_expand_kernel(
    const uint32_t* __restrict__ order, const int4* __restrict__ rects, const SortCtl* __restrict__ ctl, int gh,
    uint32_t n_chunks, int warps_per_block, uint2* __restrict__ prect, uint32_t* __restrict__ table_r,
    uint2* __restrict__ row_rec) {
  pdl_prologue();
  extern __shared__ uint32_t xp_smem[];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t chunk = blockIdx.x * (uint32_t)warps_per_block + warp;
  if (chunk >= n_chunks) return;
  // capacity overflow: only the counts are taken.  A failed sort (overflow == 2) left `order` undefined: nothing of it is
  // read and every count is written as zero, so that the scan and the plan that follow work on defined numbers.
  const uint32_t ov = ctl->overflow;
  if (ov && !kCount) return;
  uint32_t* cnt = xp_smem + (size_t)warp * (gh + 1);
  const uint32_t nvis = ov == 2u ? 0u : ctl->nvis;
  const uint32_t k0 = chunk * (uint32_t)XP_CHUNK;
  for (int b = lane; b <= gh; b += 32) cnt[b] = (kCount || b == gh) ? 0u : table_r[(size_t)b * n_chunks + chunk];
  __syncwarp();
  if (k0 < nvis) {
    const uint32_t k1 = min(k0 + (uint32_t)XP_CHUNK, nvis);
    // all loads of the chunk are issued before the first group is processed (XP_GROUPS items per lane)
    uint32_t id[XP_GROUPS], xx[XP_GROUPS], yy[XP_GROUPS];
#pragma unroll
    for (int u = 0; u < XP_GROUPS; u++) {
      const uint32_t k = k0 + 32 * u + lane;
      id[u] = k < k1 ? order[k] : 0u;
    }
#pragma unroll
    for (int u = 0; u < XP_GROUPS; u++) {
      const uint32_t k = k0 + 32 * u + lane;
      xx[u] = 0; yy[u] = 0;
      if (k < k1) {
        if (kCount) {
          const int4 r = rects[id[u]];
          xx[u] = (uint32_t)r.x | ((uint32_t)r.z << 16);
          yy[u] = (uint32_t)r.y | ((uint32_t)r.w << 16);
        } else {
          const uint2 p = prect[k];
          xx[u] = p.x; yy[u] = p.y;
        }
      }
    }
#pragma unroll
    for (int u = 0; u < XP_GROUPS; u++) {
      const uint32_t k = k0 + 32 * u + lane;
      if (k0 + 32 * u >= k1) break;
      const int lo = (int)(yy[u] & 0xffffu), hi = (int)(yy[u] >> 16);  // empty interval for lanes past the end
      if (kCount) {
        if (k < k1) prect[k] = make_uint2(xx[u], yy[u]);
        xp_count_group(lo, hi, cnt);
      } else {
        xp_emit_group<2>(lo, hi, id[u], xx[u], cnt, lane, reinterpret_cast<uint32_t*>(row_rec));
      }
    }
  }
  if (kCount) {
    __syncwarp();
    xp_counts_to_table(cnt, gh, lane, table_r + chunk, n_chunks);
  }
}

// Plan of the column expansion: records per row -> chunks per row -> chunk_base (exclusive scan over
// rows).  One block.  row_start[r] = position of row r's first record in row_rec (r = 0..gh).
__global__ void __launch_bounds__(1024) plan_kernel(const uint32_t* __restrict__ table_r, uint32_t n_chunks_r, int gh,
                                                    int gw, uint32_t* __restrict__ row_start,
                                                    uint32_t* __restrict__ chunk_base, SortCtl* __restrict__ ctl) {
  pdl_prologue();
  __shared__ uint32_t part[1024];
  const int per = (gh + 1023) / 1024;
  const int b = threadIdx.x * per, e = min(gh, b + per);
  uint32_t s = 0;
  for (int r = b; r < e; r++) {
    const uint32_t st = table_r[(size_t)r * n_chunks_r], en = table_r[(size_t)(r + 1) * n_chunks_r];
    row_start[r] = st;
    s += (en - st + XP_CHUNK - 1) / XP_CHUNK;
  }
  part[threadIdx.x] = s;
  __syncthreads();
  for (int o = 1; o < 1024; o <<= 1) {
    const uint32_t v = threadIdx.x >= o ? part[threadIdx.x - o] : 0;
    __syncthreads();
    part[threadIdx.x] += v;
    __syncthreads();
  }
  uint32_t run = part[threadIdx.x] - s;
  for (int r = b; r < e; r++) {
    const uint32_t st = table_r[(size_t)r * n_chunks_r], en = table_r[(size_t)(r + 1) * n_chunks_r];
    chunk_base[r] = run;
    run += (en - st + XP_CHUNK - 1) / XP_CHUNK;
  }
  if (threadIdx.x == 1023) {
    const uint32_t total = part[1023];
    chunk_base[gh] = total;
    row_start[gh] = table_r[(size_t)gh * n_chunks_r];
    ctl->n_chunks_c = ctl->overflow ? 0u : total;
    ctl->n_table_c = ctl->overflow ? 0u : total * (uint32_t)gw;
  }
}

// S3: column expansion.  Chunk g lies in row r (chunk_base[r] <= g < chunk_base[r+1]); its records cover
// columns [x0, x1).  Table index of (r, tx, c) = gw * chunk_base[r] + tx * nchunk_r + c, so that a linear
// exclusive scan of the table runs over tiles in row-major order and over chunks within a tile.
template <bool kCount>
__global__ void __launch_bounds__(32 * XP_MAX_WARPS) col_expand_kernel(
    const uint2* __restrict__ row_rec, const uint32_t* __restrict__ row_start, const uint32_t* __restrict__ chunk_base,
    const SortCtl* __restrict__ ctl, int gw, int gh, int warps_per_block, uint32_t* __restrict__ table_c,
    uint32_t* __restrict__ sorted_ids) {
  pdl_prologue();
  extern __shared__ uint32_t xp_smem[];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t g = blockIdx.x * (uint32_t)warps_per_block + warp;
  if (g >= ctl->n_chunks_c) return;
  uint32_t* cnt = xp_smem + (size_t)warp * (gw + 1);
  // row of this chunk: the last r with chunk_base[r] <= g
  int lo_r = 0, hi_r = gh;  // invariant: chunk_base[lo_r] <= g < chunk_base[hi_r]
  while (hi_r - lo_r > 1) {
    const int mid = (lo_r + hi_r) >> 1;
    if (chunk_base[mid] <= g) lo_r = mid; else hi_r = mid;
  }
  const int r = lo_r;
  const uint32_t cb = chunk_base[r], nch = chunk_base[r + 1] - cb, c = g - cb;
  const uint32_t j0 = row_start[r] + c * (uint32_t)XP_CHUNK;
  const uint32_t j1 = min(j0 + (uint32_t)XP_CHUNK, row_start[r + 1]);
  uint32_t* tab = table_c + (size_t)gw * cb + c;
  for (int b = lane; b <= gw; b += 32) cnt[b] = (kCount || b == gw) ? 0u : tab[(size_t)b * nch];
  __syncwarp();
  uint2 rec[XP_GROUPS];  // all records of the chunk are loaded before the first group is processed
#pragma unroll
  for (int u = 0; u < XP_GROUPS; u++) {
    const uint32_t j = j0 + 32 * u + lane;
    rec[u] = j < j1 ? row_rec[j] : make_uint2(0u, 0u);
  }
#pragma unroll
  for (int u = 0; u < XP_GROUPS; u++) {
    if (j0 + 32 * u >= j1) break;
    const int lo = (int)(rec[u].y & 0xffffu), hi = (int)(rec[u].y >> 16);
    if (kCount) xp_count_group(lo, hi, cnt);
    else xp_emit_group<1>(lo, hi, rec[u].x, 0u, cnt, lane, sorted_ids);
  }
  if (kCount) {
    __syncwarp();
    xp_counts_to_table(cnt, gw, lane, tab, nch);
  }
}

// Tile ranges from the scanned column table: start(t) = scan value of (r, tx, chunk 0); a row without
// records has no table entries and all its tiles start (and end) where the next row's first tile starts.
__global__ void __launch_bounds__(256) tile_ranges_kernel(const uint32_t* __restrict__ table_c,
                                                          const uint32_t* __restrict__ chunk_base,
                                                          SortCtl* __restrict__ ctl, int gw, int gh,
                                                          uint32_t* __restrict__ tile_ranges) {
  pdl_prologue();
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  const int ntiles = gw * gh;
  if (t >= ntiles) return;
  if (ctl->overflow) {
    if (t == 0 && ctl->overflow == 2u) ctl->R = ~0ull;  // a look-back gave up: reported as R = UINT64_MAX
    tile_ranges[2 * t] = 0;
    tile_ranges[2 * t + 1] = 0;
    atomicAdd(&ctl->class_count[0], 1u);
    return;
  }
  uint32_t se[2];
#pragma unroll
  for (int q = 0; q < 2; q++) {
    const int tt = t + q;
    size_t idx;
    if (tt >= ntiles) idx = ctl->n_table_c;
    else {
      const int r = tt / gw, tx = tt % gw;
      const uint32_t cb = chunk_base[r], nch = chunk_base[r + 1] - cb;
      idx = (size_t)gw * cb + (size_t)tx * nch;
    }
    se[q] = table_c[idx];
  }
  tile_ranges[2 * t] = se[0];
  tile_ranges[2 * t + 1] = se[1];
  atomicAdd(&ctl->class_count[length_class(se[1] - se[0])], 1u);
}

// Scheduling hint: tiles in order of non-increasing list-length class (the order within a class is whatever
// the atomics give; it affects scheduling only).  Every block rebuilds the 257 class bases in shared memory.
__global__ void __launch_bounds__(256) tile_order_kernel(const uint32_t* __restrict__ tile_ranges, SortCtl* __restrict__ ctl,
                                                         int ntiles, uint32_t* __restrict__ tile_order) {
  pdl_prologue();
  __shared__ uint32_t base[TO_CLASSES];
  if (threadIdx.x == 0) {
    uint32_t run = 0;
    for (int c = TO_CLASSES - 1; c >= 0; c--) { base[c] = run; run += ctl->class_count[c]; }
  }
  __syncthreads();
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= ntiles) return;
  const uint32_t c = length_class(tile_ranges[2 * t + 1] - tile_ranges[2 * t]);
  tile_order[base[c] + atomicAdd(&ctl->class_cursor[c], 1u)] = (uint32_t)t;
}

struct Layout {
  size_t ctl, keysA, valsA, keysB, valsB, status, sums, prect, table_r, row_start, chunk_base, row_rec, table_c, total;
  int nblk_sort;          // blocks of a radix pass over N
  uint32_t n_chunks_r;    // warps of the row expansion
  uint32_t max_chunks_c;  // upper bound of the warps of the column expansion
  uint32_t max_scan_blocks;
};

inline size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }

Layout make_layout(int64_t N, int gw, int gh, uint64_t Rcap) {
  Layout L;
  const size_t n = (size_t)N, r = (size_t)Rcap;
  L.nblk_sort = (int)((n + RS_TILE - 1) / RS_TILE);
  L.n_chunks_r = (uint32_t)((n + XP_CHUNK - 1) / XP_CHUNK);
  L.max_chunks_c = (uint32_t)(r / XP_CHUNK + (size_t)gh);
  const size_t tn = (size_t)RS_BINS * L.nblk_sort, tr = (size_t)gh * L.n_chunks_r, tc = (size_t)gw * L.max_chunks_c;
  size_t tmax = tr;
  if (tc > tmax) tmax = tc;
  L.max_scan_blocks = (uint32_t)((tmax + SCAN_BLK - 1) / SCAN_BLK + 1);
  size_t o = 0;
  L.ctl = o; o = align256(o + sizeof(SortCtl));
  L.keysA = o; o = align256(o + 4 * n);
  L.valsA = o; o = align256(o + 4 * n);
  L.keysB = o; o = align256(o + 4 * n);
  L.valsB = o; o = align256(o + 4 * n);
  L.status = o; o = align256(o + 8 * 4 * tn);  // look-back status words of the four radix passes
  L.sums = o; o = align256(o + 4 * (size_t)L.max_scan_blocks);
  L.prect = o; o = align256(o + 8 * n);
  L.table_r = o; o = align256(o + 4 * (tr + 1));
  L.row_start = o; o = align256(o + 4 * (size_t)(gh + 1));
  L.chunk_base = o; o = align256(o + 4 * (size_t)(gh + 1));
  L.row_rec = o; o = align256(o + 8 * r);
  L.table_c = o; o = align256(o + 4 * (tc + 1));
  L.total = o;
  return L;
}

// Warps per block of an expansion sweep with `bins` uint32 counters per warp in dynamic shared memory.
inline int xp_warps(int bins) {
  int w = (int)((160 * 1024) / ((size_t)bins * 4));
  if (w > XP_MAX_WARPS) w = XP_MAX_WARPS;
  if (w < 1) w = 1;
  return w;
}

// Launch `kernel` on `st` so that it may overlap the tail of the kernel before it in the stream (see pdl_prologue).
template <typename... P, typename... A>
cudaError_t launch_chained(void (*kernel)(P...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, A... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid;
  cfg.blockDim = block;
  cfg.dynamicSmemBytes = smem;
  cfg.stream = st;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
#ifdef MG_NO_PDL
  cfg.attrs = nullptr;
  cfg.numAttrs = 0;
#else
  cfg.attrs = attr;
  cfg.numAttrs = 1;
#endif
  return cudaLaunchKernelEx(&cfg, kernel, static_cast<P>(args)...);
}

template <typename K>
int xp_prepare(K kernel, size_t smem) {
  if (smem > 48 * 1024) MG_CHECK_CUDA(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  return MG_OK;
}

int scan_table(uint32_t* table, uint32_t n_static, const uint32_t* n_dev, uint32_t n_max, uint32_t* sums, cudaStream_t st) {
  const uint32_t nb = (n_max + SCAN_BLK - 1) / SCAN_BLK;
  const uint32_t grid = nb ? nb : 1;
  MG_CHECK_CUDA(launch_chained(scan_sums_kernel, dim3(grid), dim3(SCAN_THREADS), (size_t)(0), st, table, n_static, n_dev, sums));
  MG_CHECK_CUDA(launch_chained(scan_apply_kernel, dim3(grid), dim3(SCAN_THREADS), (size_t)(0), st, table, n_static, n_dev, sums));
  MG_CHECK_LAUNCH();
  return MG_OK;
}

}  // namespace

extern "C" size_t mg_workspace_bytes(int64_t N, int32_t width, int32_t height, uint64_t R_capacity) {
  if (N < 0 || width <= 0 || height <= 0 || R_capacity >= (1ull << 32)) return 0;
  const int gw = (width + MG_TILE - 1) / MG_TILE, gh = (height + MG_TILE - 1) / MG_TILE;
  return make_layout(N, gw, gh, R_capacity).total;
}

#ifdef MG_TESTING
extern "C" void mg_debug_set_lookback_spin_limit(int polls) { g_spin_limit.store(polls < 0 ? LB_SPIN_LIMIT : polls); }
#endif

extern "C" int mg_bin_sort(const mg_camera* cam, int64_t N, const float* depths, const int32_t* rects,
                           const uint32_t* tiles_touched, uint64_t R_capacity, void* workspace, size_t workspace_bytes,
                           uint32_t* sorted_ids, uint32_t* tile_ranges, uint32_t* tile_order, uint64_t* R_out_host,
                           void* stream) {
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
  unsigned long long* status = (unsigned long long*)(ws + L.status);
  uint32_t* sums = (uint32_t*)(ws + L.sums);
  uint2* prect = (uint2*)(ws + L.prect);
  uint32_t* table_r = (uint32_t*)(ws + L.table_r);
  uint32_t *row_start = (uint32_t*)(ws + L.row_start), *chunk_base = (uint32_t*)(ws + L.chunk_base);
  uint2* row_rec = (uint2*)(ws + L.row_rec);
  uint32_t* table_c = (uint32_t*)(ws + L.table_c);

  MG_CHECK_CUDA(cudaMemsetAsync(ctl, 0, sizeof(SortCtl), st));
  if (N == 0) {
    MG_CHECK_CUDA(cudaMemsetAsync(tile_ranges, 0, sizeof(uint32_t) * 2 * (size_t)gw * gh, st));
    if (tile_order) {
      MG_CHECK_CUDA(launch_chained(tile_order_kernel, dim3((gw * gh + 255) / 256), dim3(256), (size_t)(0), st, tile_ranges, ctl, gw * gh, tile_order));
      MG_CHECK_LAUNCH();
    }
    if (R_out_host) MG_CHECK_CUDA(cudaMemcpyAsync(R_out_host, &ctl->R, sizeof(uint64_t), cudaMemcpyDeviceToHost, st));
    return MG_OK;
  }

  // S1: depth order of the N Gaussians (culled ones last), R, nvis, overflow flag, digit histograms
  static MgOncePerDevice attr_set;  // function attributes belong to a device
  int dev = 0, sms = 0;
  if (int rc = mg_current_device(&dev, &sms)) return rc;
  if (!attr_set.is_done(dev)) {
    MG_CHECK_CUDA(cudaFuncSetAttribute(radix_onesweep_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(RadixSmem)));
    MG_CHECK_CUDA(cudaFuncSetAttribute(radix_onesweep_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(RadixSmem)));
    attr_set.set_done(dev);
  }
  const int dk_grid = sms * 8;
#ifdef MG_TESTING
  const int spin_limit = g_spin_limit.load(std::memory_order_relaxed);
#else
  const int spin_limit = LB_SPIN_LIMIT;
#endif
  MG_CHECK_CUDA(cudaMemsetAsync(status, 0, sizeof(unsigned long long) * 4 * (size_t)L.nblk_sort * RS_BINS, st));
  {
    const int64_t want = (N + 255) / 256;
    MG_CHECK_CUDA(launch_chained(depth_hist_kernel, dim3((unsigned)(want < dk_grid ? want : dk_grid)), dim3(256), (size_t)(0), st, N, depths, tiles_touched, ctl));
  }
  MG_CHECK_CUDA(launch_chained(ctl_finalize_kernel, dim3(1), dim3(RS_BINS), (size_t)(0), st, ctl, (unsigned long long)R_capacity));
  MG_CHECK_LAUNCH();
  {
    // pass 0 reads the caller's depths and tiles_touched and writes the visible (key, index) pairs to B; then B -> A -> B -> A
    MG_CHECK_CUDA(launch_chained(radix_onesweep_kernel<true>, dim3(L.nblk_sort), dim3(RS_THREADS), (size_t)(sizeof(RadixSmem)), st, 
        reinterpret_cast<const uint32_t*>(depths), tiles_touched, keysB, valsB, (uint32_t)N, 0, ctl, status, spin_limit));
    MG_CHECK_LAUNCH();
    const uint32_t *ki = keysB, *vi = valsB;
    uint32_t *ko = keysA, *vo = valsA;
    for (int pass = 1; pass < 4; pass++) {
      MG_CHECK_CUDA(launch_chained(radix_onesweep_kernel<false>, dim3(L.nblk_sort), dim3(RS_THREADS), (size_t)(sizeof(RadixSmem)), st, 
          ki, vi, ko, vo, (uint32_t)N, pass, ctl, status + (size_t)pass * L.nblk_sort * RS_BINS, spin_limit));
      MG_CHECK_LAUNCH();
      const uint32_t *tk = ki, *tv = vi;
      ki = ko; vi = vo;
      ko = const_cast<uint32_t*>(tk); vo = const_cast<uint32_t*>(tv);
    }
  }
  const uint32_t* order = valsA;  // after 4 passes the result is in (keysA, valsA)

  // S2: row expansion
  {
    const int wpb = xp_warps(gh + 1);
    const size_t smem = (size_t)wpb * (gh + 1) * 4;
    if (int rc = xp_prepare(row_expand_kernel<true>, smem)) return rc;
    if (int rc = xp_prepare(row_expand_kernel<false>, smem)) return rc;
    const unsigned grid = (L.n_chunks_r + wpb - 1) / wpb;
    const uint32_t tr = (uint32_t)gh * L.n_chunks_r;
    MG_CHECK_CUDA(launch_chained(row_expand_kernel<true>, dim3(grid), dim3(32 * wpb), (size_t)(smem), st, order, (const int4*)rects, ctl, gh, L.n_chunks_r, wpb, prect, table_r, row_rec));
    if (int rc = scan_table(table_r, tr, nullptr, tr, sums, st)) return rc;
    MG_CHECK_CUDA(launch_chained(plan_kernel, dim3(1), dim3(1024), (size_t)(0), st, table_r, L.n_chunks_r, gh, gw, row_start, chunk_base, ctl));
    MG_CHECK_CUDA(launch_chained(row_expand_kernel<false>, dim3(grid), dim3(32 * wpb), (size_t)(smem), st, order, (const int4*)rects, ctl, gh, L.n_chunks_r, wpb, prect, table_r, row_rec));
    MG_CHECK_LAUNCH();
  }
  // S3: column expansion and tile ranges
  {
    const int wpb = xp_warps(gw + 1);
    const size_t smem = (size_t)wpb * (gw + 1) * 4;
    if (int rc = xp_prepare(col_expand_kernel<true>, smem)) return rc;
    if (int rc = xp_prepare(col_expand_kernel<false>, smem)) return rc;
    const unsigned grid = (L.max_chunks_c + wpb - 1) / wpb;
    const uint32_t tc_max = (uint32_t)gw * L.max_chunks_c;
    MG_CHECK_CUDA(launch_chained(col_expand_kernel<true>, dim3(grid), dim3(32 * wpb), (size_t)(smem), st, row_rec, row_start, chunk_base, ctl, gw, gh, wpb, table_c, sorted_ids));
    if (int rc = scan_table(table_c, 0, &ctl->n_table_c, tc_max, sums, st)) return rc;
    MG_CHECK_CUDA(launch_chained(col_expand_kernel<false>, dim3(grid), dim3(32 * wpb), (size_t)(smem), st, row_rec, row_start, chunk_base, ctl, gw, gh, wpb, table_c, sorted_ids));
    MG_CHECK_CUDA(launch_chained(tile_ranges_kernel, dim3((gw * gh + 255) / 256), dim3(256), (size_t)(0), st, table_c, chunk_base, ctl, gw, gh, tile_ranges));
    if (tile_order) MG_CHECK_CUDA(launch_chained(tile_order_kernel, dim3((gw * gh + 255) / 256), dim3(256), (size_t)(0), st, tile_ranges, ctl, gw * gh, tile_order));
    MG_CHECK_LAUNCH();
  }
  if (R_out_host) MG_CHECK_CUDA(cudaMemcpyAsync(R_out_host, &ctl->R, sizeof(uint64_t), cudaMemcpyDeviceToHost, st));
  return MG_OK;
}
