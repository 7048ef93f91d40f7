/* mg.h -- C-ABI of libmg: masked rasterization of 3D Gaussians (MaskGaussian, arXiv 2412.20522)
 * for NVIDIA B200 (sm_100a).  Citations "PAPER.md:n" are lines of the paper text; "reading k" is a
 * row of DESIGN.md's table of readings (where the paper is silent).
 *
 * One training-iteration pass of the hot path is five calls, in this order:
 *
 *   mg_preprocess      splat every Gaussian, masks NOT consulted  (PAPER.md:64-66 sec. 3.1; :30, :78)
 *   mg_bin_sort        per-tile depth-ordered lists                (PAPER.md:66 "depth order"; :74 16x16 tiles)
 *   mg_render_fwd      masked blend, Eq. 3-4 + background Eq. 9-10
 *   mg_render_bwd      reverse traversal, Eq. 11-18 -> dL/dM_i and the usual gradients
 *   mg_preprocess_bwd  chain rule through the projection           (implied by PAPER.md:156)
 *
 * Conventions
 *   - Every call returns 0 (MG_OK) or a negative mg_status; mg_last_error_string() describes the last
 *     failure on the calling thread.  No exceptions cross the boundary.
 *   - Every array pointer is a DEVICE pointer unless its name ends in _host (pinned or pageable HOST
 *     memory written asynchronously: valid after the stream is synchronised).  `cam` is a HOST pointer,
 *     read during the call.  The caller owns every buffer; the library allocates nothing persistent.
 *   - `stream` is a cudaStream_t (NULL = default stream).  All work is enqueued on it; calls are
 *     asynchronous.
 *     Calls may overlap on different streams, and be issued from different host threads, as long as they
 *     share no output or scratch buffer: the library keeps no device-side state of its own (every counter
 *     lives in caller memory) and its per-device one-time initialisations are thread-safe.  The one exception
 *     is mg_render_loss_static, whose scratch is an array inside the library: see there.
 *   - Domain: finite inputs; quats need not be unit but |q|^2 must be a normal fp32 number (1e-19 < |q| < 1e19) --
 *     a zero quaternion has no rotation, its covariance is not a number and the Gaussian is culled (radius 0, exact
 *     zeros everywhere), and a norm that under- or overflows in fp32 behaves the same; exp(log_scale) and the projected
 *     covariance must stay finite in fp32 (scales below ~1e15 pixels): beyond that the Gaussian is culled likewise.
 *   - Layouts: packed row-major fp32.  means[N][3], log_scales[N][3], quats[N][4] as (w,x,y,z),
 *     opacity_logits[N], sh[N][K][3] with K=(sh_degree+1)^2 (coefficient-major, RGB innermost),
 *     masks[N] (any real value; tests use {0,1}; Eq. 4 is affine in M), images planar [3][H][W].
 *     Float arrays must be 16-byte aligned (cudaMalloc / torch allocations are).
 *   - Gradient outputs are OVERWRITTEN (never accumulated into caller content).  Culled Gaussians get
 *     exact zeros everywhere, including dL_dmask.
 */
#ifndef MG_H_
#define MG_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* Constants of the method (readings 1, 11-14; the paper states none of them). */
#define MG_TILE 16              /* PAPER.md:74 "tile (16x16 grid)" */
#define MG_ALPHA_MIN (1.0f / 255.0f) /* a pair with alpha < 1/255 is skipped (mask not consulted) */
#define MG_ALPHA_MAX 0.99f      /* alpha = min(0.99, o * G) */
#define MG_T_MIN 1e-4f          /* a pixel stops before the entry that would take T below 1e-4 */
#define MG_DILATION 0.3f        /* low-pass added to the diagonal of the 2D covariance */
#define MG_ZNEAR 0.2f           /* Gaussians with camera-space z <= 0.2 are culled */
#define MG_JCLAMP 1.3f          /* x/z, y/z clamped to +-1.3*W/(2fx), +-1.3*H/(2fy) inside the Jacobian */
#define MG_EIG_FLOOR 0.1f       /* floor under the square root of the eigenvalue formula */

typedef enum {
  MG_OK = 0,
  MG_ERR_INVALID_ARG = -1, /* null pointer, negative size, sh_degree outside 0..3, image larger than 2^15 tiles per side */
  MG_ERR_CAPACITY = -2,    /* caller buffer or workspace too small */
  MG_ERR_CUDA = -3         /* a CUDA call failed; see mg_last_error_string() */
} mg_status;

typedef struct {
  int32_t width, height;
  float fx, fy, cx, cy; /* pinhole intrinsics in pixels; pixel (i,j) has its centre at (i+0.5, j+0.5) (reading 15) */
  float R[9];           /* world->camera rotation, row-major: x_cam = R x_world + t; camera looks down +z, x right, y down */
  float t[3];
  float bg[3];          /* background colour c_bg (Eq. 10) */
  int32_t sh_degree;    /* 0..3 */
} mg_camera;

const char* mg_last_error_string(void);
int mg_version(void);

/* Bytes of device scratch mg_bin_sort needs for N Gaussians, a width x height image and at most
 * R_capacity duplicated keys.  Returns 0 on invalid arguments. */
size_t mg_workspace_bytes(int64_t N, int32_t width, int32_t height, uint64_t R_capacity);

/* Step a1-a3.  Per Gaussian: s = exp(log_scale), q/|q|, o = sigmoid(logit);
 * camera-space mean, cull z <= MG_ZNEAR; Sigma = Rot S^2 Rot^T; Sigma2D = J W Sigma W^T J^T + 0.3 I;
 * conic = Sigma2D^-1; projected centre; colour = max(0, 0.5 + sum_j Y_j(dir) sh_j); radius =
 * ceil(3 sqrt(lambda_max)); rectangle of 16x16 tiles touched.  Masks are not an argument: "all
 * Gaussians are splatted without any attribute masked out".
 * Outputs (culled Gaussians: zeros, radii = 0, tiles_touched = 0):
 *   means2d[N][2] pixel-index coordinates; depths[N] camera z; conic_opacity[N][4] = (A, B, C, o) with
 *   power = -1/2 (A dx^2 + 2 B dx dy + C dy^2); rgb[N][3]; radii[N]; rects[N][4] = (x0, y0, x1, y1) in
 *   tile units, max exclusive; tiles_touched[N]; clamped[N] bit k = colour channel k clamped at 0.
 *   num_rendered (DEVICE, one uint64, may be NULL): overwritten with R = sum of tiles_touched.
 *   num_rendered_host (may be NULL; needs num_rendered): a copy of it, written asynchronously. */
int mg_preprocess(const mg_camera* cam, int64_t N, const float* means, const float* log_scales, const float* quats,
                  const float* opacity_logits, const float* sh, float* means2d, float* depths, float* conic_opacity,
                  float* rgb, int32_t* radii, int32_t* rects, uint32_t* tiles_touched, uint8_t* clamped,
                  uint64_t* num_rendered, uint64_t* num_rendered_host, void* stream);

/* Step a4-a6.  Result = the duplicated (tile, depth) keys in ascending order of the
 * 64-bit key (tile_id << 32 | fp32 bits of depth), ties by Gaussian index, tile_id = ty * gw + tx:
 *   sorted_ids[R]       Gaussian index of each sorted key
 *   tile_ranges[gw*gh][2] = [start, end) of each tile in sorted_ids (start == end for an empty tile)
 *   tile_order[gw*gh] (may be NULL): a scheduling hint for the two render calls -- a permutation of the tile
 *                       ids in which the length class of the tile lists never increases (class(0) = 0,
 *                       class(n) = 1 + 8 floor(log2 n) + the next 3 bits of n), so that a grid launched in this
 *                       order starts its longest tiles first.  The order within a class is unspecified.
 *   R_out_host (may be NULL): the true R, written asynchronously.
 * R must be < 2^32.  If R > R_capacity nothing is written to sorted_ids, every tile range is set to
 * [0, 0) and *R_out_host (> R_capacity) tells the caller to retry with larger buffers.
 * Internal failure: the radix passes chain their blocks through look-backs that poll a predecessor's status
 * word; a poll that exhausts its limit (impossible in a correct run: a predecessor is always resident) does
 * not return a wrong order: nothing is emitted, every tile range is [0, 0) and *R_out_host = UINT64_MAX.
 * workspace: at least mg_workspace_bytes(N, W, H, R_capacity) bytes, 256-byte aligned. */
int mg_bin_sort(const mg_camera* cam, int64_t N, const float* depths, const int32_t* rects,
                const uint32_t* tiles_touched, uint64_t R_capacity, void* workspace, size_t workspace_bytes,
                uint32_t* sorted_ids, uint32_t* tile_ranges, uint32_t* tile_order, uint64_t* R_out_host,
                void* stream);

/* Test hook (failure injection), NOT part of the shipped ABI: it exists only in the test build of the library
 * (libmg_testing.so, compiled with -DMG_TESTING); libmg.so neither exports it nor has the state behind it.
 * polls a look-back makes before it gives up; 0 = every look-back after a call's first tile gives up at once,
 * negative = the default (2^26).  Process-wide in that build: not for use next to concurrent mg_bin_sort calls. */
#ifdef MG_TESTING
void mg_debug_set_lookback_spin_limit(int polls);
#endif

/* Step a7 (Eq. 3-4; Eq. 9-10).  Per pixel, front to back over its tile's
 * list: alpha = min(0.99, o G); skip if power > 0 or alpha < 1/255 (mask NOT consulted, reading 2);
 * a = M alpha; T' = T (1 - a); stop if T' < 1e-4 (this entry is not blended, reading 3-4);
 * C += a T c; T = T'.  Then image = C + T c_bg.
 *   image[3][H][W]; final_T[H][W] = T_{N+1}; n_contrib[H][W] = the number of list entries the pixel
 *   consumed: the entries in front of the one that stopped it, or the length of the tile's list if nothing
 *   stopped it (reading 5).  It bounds the reverse traversal: every entry that contributed to the pixel,
 *   masked or not, lies at a 1-based position <= n_contrib, and no entry at or behind the stop does.  The
 *   forward pass therefore never has to look at an entry with M = 0.
 *   tile_order (may be NULL = row-major): the order in which tiles are scheduled (mg_bin_sort's hint); it has
 *   no effect on any output. */
int mg_render_fwd(const mg_camera* cam, const uint32_t* sorted_ids, const uint32_t* tile_ranges,
                  const uint32_t* tile_order, const float* means2d, const float* conic_opacity, const float* rgb, const float* masks,
                  float* image, float* final_T, uint32_t* n_contrib, void* stream);

/* Step a8 (Eq. 11, 13-18).  Per pixel, from its last contributor back to the front:
 * T_i = T_{i+1} / (1 - a_i); b by the recursion of Eq. 11; dL/dM_i by Eq. 18 (including the background
 * term); dL/dalpha_i = M_i * (same bracket); chain to colour, opacity (w.r.t. the activated o), conic and
 * projected centre (pixels).  Zero gradient to (o, conic, centre) where the 0.99 clamp is active
 * (reading 6).  A masked Gaussian (M = 0) gets dL/dM only (Fig. 1).
 * Sums over pixels use fp32 atomics: results vary in the last bits from run to run.
 * tile_order: as for mg_render_fwd. */
int mg_render_bwd(const mg_camera* cam, int64_t N, const uint32_t* sorted_ids, const uint32_t* tile_ranges,
                  const uint32_t* tile_order, const float* means2d, const float* conic_opacity, const float* rgb, const float* masks,
                  const float* final_T, const uint32_t* n_contrib, const float* dL_dimage, float* dL_dmeans2d,
                  float* dL_dconic, float* dL_dopacity, float* dL_drgb, float* dL_dmask, void* stream);

/* Step a9.  Vector-Jacobian product of mg_preprocess: from (dL_dmeans2d[N][2], dL_dconic[N][3] for
 * (A,B,C), dL_dopacity[N], dL_drgb[N][3]) to gradients w.r.t. the raw inputs: dL_dmeans[N][3],
 * dL_dlog_scales[N][3], dL_dquats[N][4] (w.r.t. the un-normalised quaternion), dL_dopacity_logits[N],
 * dL_dsh[N][K][3].  No gradient flows through depth, radius or rect; none through a clamped colour
 * channel.  radii and clamped are mg_preprocess's outputs for the same inputs and camera. */
int mg_preprocess_bwd(const mg_camera* cam, int64_t N, const float* means, const float* log_scales,
                      const float* quats, const float* opacity_logits, const float* sh, const int32_t* radii,
                      const uint8_t* clamped, const float* dL_dmeans2d, const float* dL_dconic,
                      const float* dL_dopacity, const float* dL_drgb, float* dL_dmeans, float* dL_dlog_scales,
                      float* dL_dquats, float* dL_dopacity_logits, float* dL_dsh, void* stream);

/* ---- The mask head around the rasterizer.  Random numbers are INPUTS: the library draws none.
 *
 * mg_mask_sample (sec. 3.3: "we assign 2 learnable mask scores for each Gaussian, and apply Gumbel-Softmax
 * to sample one differentiable category out of the 2 scores, denoted M_i in {0,1}").  scores[N][2], uniforms[N][2] in
 * (0,1).  A uniform outside the open interval -- generators on [0,1) return exactly 0, rounding to fp32 can give exactly
 * 1 -- is taken as the nearest fp32 value inside it: u is clamped to [2^-126, 1 - 2^-24] (reading 29), so the
 * noise lies in [-4.47, 16.64] and every output is finite; NaN uniforms are outside the contract.  The same holds for
 * mg_mask_prune_keep.  g = -log(-log u); d = (s_1 + g_1) - (s_0 + g_0); masks[i] = 1 if d > 0 else 0 (category 1 = present, a tie
 * gives 0); soft[i] (may be NULL) = softmax((s + g) / tau)_1 = sigmoid(d / tau), kept for the backward pass.
 * tau > 0 is not stated in the paper (reading 22). */
int mg_mask_sample(int64_t N, const float* scores, const float* uniforms, float tau, float* masks, float* soft,
                   void* stream);

/* Straight-through gradient of the hard sample (reading 23): dL_dscores[i] = (-t, t), t = dL_dmask[i] y (1 - y) / tau,
 * y = soft[i].  dL_dscores[N][2] is overwritten. */
int mg_mask_sample_bwd(int64_t N, const float* soft, const float* dL_dmask, float tau, float* dL_dscores, void* stream);

/* Eq. 7-8: L_m = (1/N sum M_i)^2, L = L_render + lambda_m L_m.  stats (DEVICE, 3 doubles, overwritten):
 * stats[0] = sum M, stats[1] = lambda_m L_m, stats[2] = mean M.  If dL_dmask is not NULL, lambda_m * 2 * mean / N is
 * ADDED to every element (it already holds dL_render/dM from mg_render_bwd). */
int mg_mask_loss(int64_t N, const float* masks, float lambda_m, float* dL_dmask, double* stats, void* stream);

/* "we sample each Gaussian 10 times and remove those that are never sampled".  uniforms[n_draws][N][2];
 * keep[i] = 1 iff M_i = 1 in at least one draw. */
int mg_mask_prune_keep(int64_t N, int32_t n_draws, const float* scores, const float* uniforms, uint8_t* keep, void* stream);

/* Stable compaction by keep[N]: for each of the n_arrays (<= 16) arrays of row_floats[a] floats per Gaussian, the rows
 * of the kept Gaussians are copied, in order, to dst[a] (capacity N rows; src and dst must not overlap).  src, dst and
 * row_floats are HOST arrays (of device pointers / ints).  *N_out_host = number kept, written asynchronously.
 * workspace: mg_compact_workspace_bytes(N) bytes of device memory, 256-byte aligned. */
size_t mg_compact_workspace_bytes(int64_t N);
int mg_compact(int64_t N, const uint8_t* keep, int32_t n_arrays, const float* const* src, float* const* dst,
               const int32_t* row_floats, void* workspace, size_t workspace_bytes, uint64_t* N_out_host, void* stream);

/* ---- The render loss.  Eq. 8: L = L_render + lambda_m L_m with L_render
 * "the original rendering loss", which the paper does not define; reading 26: the loss of the 3DGS method the paper
 * modifies, L_render = (1 - lambda) mean|I - G| + lambda (1 - mean SSIM(I, G)), SSIM per channel with a
 * separable 11-tap Gaussian window (sigma 1.5, normalised), zero padding, C1 = 0.01^2, C2 = 0.03^2, means over all
 * 3 H W elements.  image, target, dL_dimage: planar [3][H][W]; dL_dimage = dL_render/dimage is overwritten.
 * stats (DEVICE, 3 doubles, overwritten): mean|I - G|, mean SSIM, L_render.
 * workspace: mg_render_loss_workspace_bytes(width, height) bytes of device memory. */
size_t mg_render_loss_workspace_bytes(int32_t width, int32_t height);
int mg_render_loss(int32_t width, int32_t height, const float* image, const float* target, float lambda_dssim,
                   float* dL_dimage, double* stats, void* workspace, size_t workspace_bytes, void* stream);

/* mg_render_loss_static: the same loss and gradient, for a caller that cannot provide a workspace because it cannot
 * allocate device memory where it needs the loss -- code running inside an application whose own memory manager claimed
 * the whole GPU at start-up and hands it only input and output buffers, a plug-in or callback bound to "no allocation
 * after initialisation", a frame loop in which the device-wide synchronisation of cudaMalloc / cudaFree is not
 * acceptable.  The call allocates and frees nothing, on the host side of CUDA or the device side: its scratch (9 floats
 * per pixel) is an array built into the library's device image.
 *   Limit: width * height <= MG_RENDER_LOSS_STATIC_MAX_PIXELS (2^21: 1920 x 1080 fits); a larger image is rejected with
 *   MG_ERR_CAPACITY and a message that names the limit -- use mg_render_loss with your own workspace then.
 *   Cost: 72 MiB of device memory (9 * 4 B * 2^21), reserved on EVERY GPU on which the CUDA runtime loads this library's
 *   code (at the latest at the first render-loss call there) and held until the process exits, whether or not
 *   mg_render_loss_static is ever called.
 *   First call on a device: looks up the array's device address (cudaGetSymbolAddress, with that device current; the
 *   result is cached per device) and uploads the filter window.  That makes the CUDA runtime load the kernels and reserve
 *   the array, so make the first call on each device during set-up, outside any stream capture and before the point from
 *   which nothing may be allocated.  Later calls only enqueue a 24-byte clear of `stats` and three kernels on `stream`.
 *   Sharing: all calls on a device use the same array, and it keeps what the last call wrote.  Nothing in it needs to
 *   start at zero (every element a call reads it has written itself), so calls of any image sizes may follow one another
 *   on one stream.  Two calls that can run on the GPU at the same time (different streams, or different host threads
 *   without ordering between their streams) RACE on it and give wrong gradients: order them, or give all but one of
 *   them mg_render_loss with a workspace.
 * image, target, dL_dimage, stats, lambda_dssim, the outputs and the error codes otherwise: exactly as mg_render_loss. */
#define MG_RENDER_LOSS_STATIC_MAX_PIXELS (1 << 21)
int mg_render_loss_static(int32_t width, int32_t height, const float* image, const float* target, float lambda_dssim,
                          float* dL_dimage, double* stats, void* stream);

/* ---- Density-control statistics and the optimiser step.  The paper keeps "the densification
 * scheme" and the training procedure of the 3DGS method it modifies and prints neither; DESIGN.md
 * readings 27-28 state what is computed.
 *
 * mg_density_stats (reading 27), after mg_render_bwd of a view: for every Gaussian with radii[i] > 0 (visible in it)
 *   grad_accum[i] += sqrt((scale_x g_x)^2 + (scale_y g_y)^2), g = dL_dmeans2d[i] (pixels, reading 19);
 *   denom[i] += 1;  max_radii[i] = max(max_radii[i], radii[i]).
 * grad_accum, denom, max_radii: [N] fp32, UPDATED IN PLACE (the caller zeroes them when a densification step has consumed
 * them); Gaussians with radii[i] == 0 are neither read nor written.  (scale_x, scale_y) = (1, 1) keeps pixel units;
 * (W/2, H/2) gives the normalised-device-coordinate units of the 3DGS lineage's thresholds. */
int mg_density_stats(int64_t N, const float* dL_dmeans2d, const int32_t* radii, float scale_x, float scale_y,
                     float* grad_accum, float* denom, float* max_radii, void* stream);

/* mg_adam_step (reading 28): Adam (Kingma & Ba 2015, Algorithm 1, bias-corrected) over up to MG_ADAM_MAX_GROUPS attribute
 * groups in ONE launch, each with its own learning rate:
 *   m <- beta1 m + (1 - beta1) g;  v <- beta2 v + (1 - beta2) g^2;
 *   p <- p - lr (m / (1 - beta1^step)) / (sqrt(v / (1 - beta2^step)) + eps),   step = 1, 2, ...
 * groups_host: HOST array of n_groups descriptors of DEVICE arrays with n_rows * row_floats floats each (16-byte aligned);
 * param, m, v are UPDATED IN PLACE, grad is read only.  fp32 state and arithmetic (IEEE sqrt and division).
 * radii (DEVICE, may be NULL): if given, every group must have one row per Gaussian (n_rows = N) and the rows of Gaussians
 * with radii[i] == 0 are left untouched -- parameter and both moments are neither decayed nor written (the variant that
 * skips Gaussians not visible in the view, whose gradient is exactly zero).  This is a choice of SEMANTICS, not a faster
 * path: the skip is per 16-byte vector, every vector still looks up its row's radius, and on the B200 the call is slower
 * than the dense step until most rows are skipped (1.22 ms against 1.04 ms with 71 % of 3 M Gaussians visible).
 * NULL = every element is updated. */
#define MG_ADAM_MAX_GROUPS 8
typedef struct {
  float* param;
  const float* grad;
  float* m;
  float* v;
  int64_t n_rows;
  int32_t row_floats; /* 1..1024 */
  float lr;
} mg_adam_group;
int mg_adam_step(int32_t n_groups, const mg_adam_group* groups_host, float beta1, float beta2, float eps, int64_t step,
                 const int32_t* radii, void* stream);

/* ---- Measurement aid (the FP32 roofline of the blend kernels needs a measured peak; the driver's
 * MEASURED_PEAKS.json has none).  Runs dependent-free FMA chains on every SM for at least min_seconds per instruction
 * form and times them with CUDA events; SYNCHRONOUS (returns when the measurement is done).
 * tflops_host (HOST, 4 doubles): [0] scalar FFMA sustained over the measurement, [1] its best round, [2] packed
 * fma.rn.f32x2 sustained, [3] its best round -- in TFLOP/s, an FMA counted as 2 flop.  scratch: one DEVICE float. */
int mg_measure_fp32_peak(double min_seconds, double* tflops_host, float* scratch, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* MG_H_ */
