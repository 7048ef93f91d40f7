// mg_common.cuh -- shared by the kernels of libmg (product code; nothing here is used by oracle/).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "mg.h"

void mg_set_error(const char* fmt, ...);

// Per-device facts and one-time initialisations (api.cu).  Thread-safe: the cache entries are atomics and every
// initialisation is idempotent, so two host threads that race on a first call both do the same harmless work.
int mg_current_device(int* dev, int* sm_count);  // MG_OK or MG_ERR_CUDA
struct MgOncePerDevice {                         // zero-initialised static: done[dev] != 0 once the init has run
  int done[64];
  bool is_done(int dev) const { return __atomic_load_n(&done[dev & 63], __ATOMIC_ACQUIRE) != 0; }
  void set_done(int dev) { __atomic_store_n(&done[dev & 63], 1, __ATOMIC_RELEASE); }
};

#define MG_CHECK_CUDA(expr)                                                              \
  do {                                                                                   \
    cudaError_t e__ = (expr);                                                            \
    if (e__ != cudaSuccess) {                                                            \
      mg_set_error("%s failed: %s (%s:%d)", #expr, cudaGetErrorString(e__), __FILE__, __LINE__); \
      return MG_ERR_CUDA;                                                                \
    }                                                                                    \
  } while (0)

#define MG_CHECK_LAUNCH() MG_CHECK_CUDA(cudaGetLastError())

#define MG_REQUIRE(cond, msg)               \
  do {                                      \
    if (!(cond)) {                          \
      mg_set_error("invalid argument: %s", msg); \
      return MG_ERR_INVALID_ARG;            \
    }                                       \
  } while (0)

static inline int mg_check_camera(const mg_camera* cam) {
  MG_REQUIRE(cam != nullptr, "cam is null");
  MG_REQUIRE(cam->width > 0 && cam->height > 0, "image size must be positive");
  MG_REQUIRE(cam->width <= (1 << 19) && cam->height <= (1 << 19), "image larger than 2^15 tiles per side");
  MG_REQUIRE(cam->sh_degree >= 0 && cam->sh_degree <= 3, "sh_degree must be 0..3");
  MG_REQUIRE(cam->fx > 0.f && cam->fy > 0.f, "focal lengths must be positive");
  return MG_OK;
}

static inline int mg_grid_w(const mg_camera* c) { return (c->width + MG_TILE - 1) / MG_TILE; }
static inline int mg_grid_h(const mg_camera* c) { return (c->height + MG_TILE - 1) / MG_TILE; }

// Real spherical-harmonics constants (Condon-Shortley sign, order l, m=-l..l; reading 16).
#define MG_SH_C0 0.28209479177387814f
#define MG_SH_C1 0.4886025119029199f
#define MG_SH_C2_0 1.0925484305920792f
#define MG_SH_C2_1 -1.0925484305920792f
#define MG_SH_C2_2 0.31539156525252005f
#define MG_SH_C2_3 -1.0925484305920792f
#define MG_SH_C2_4 0.5462742152960396f
#define MG_SH_C3_0 -0.5900435899266435f
#define MG_SH_C3_1 2.890611442640554f
#define MG_SH_C3_2 -0.4570457994644658f
#define MG_SH_C3_3 0.3731763325901154f
#define MG_SH_C3_4 -0.4570457994644658f
#define MG_SH_C3_5 1.445305721320277f
#define MG_SH_C3_6 -0.5900435899266435f

// ---- asynchronous 16-byte copies global -> shared (LDGSTS): no registers are held while the data is in flight, so a
// thread can have many more of them outstanding than loads into registers.  .ca (allocate at every level, like the loads
// these copies replace), not .cg: with .cg the kernel itself was 4 us faster still, but the mg_preprocess that follows it
// in the next frame ran 18 us slower (measured in the frame) -- what a kernel leaves in the caches is
// part of its cost.
#ifdef __CUDACC__
__device__ __forceinline__ void mg_cp_async16(void* smem_dst, const void* gmem_src) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"((uint32_t)__cvta_generic_to_shared(smem_dst)), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void mg_cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void mg_cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }
#endif
