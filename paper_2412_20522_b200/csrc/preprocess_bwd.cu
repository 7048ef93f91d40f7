// preprocess_bwd.cu -- mg_preprocess_bwd: vector-Jacobian product of mg_preprocess (step a9).
// The paper gives no formulas for this step ("We modify the CUDA rasterization code of 3DGS",
// PAPER.md:156); it is the chain rule of DESIGN.md O1-O8, hand-derived here in reverse mode.  The
// oracle obtains the same quantity by forward-mode dual numbers, so the two derivations are independent.
// HBM-bound: one thread per Gaussian; 236 B of inputs + 36 B of upstream gradients in, 236 B out;
// the 192-byte SH rows (in and out) are staged through shared memory so that global accesses coalesce.
#include "mg_common.cuh"

namespace {

// SH rows move through shared memory: a warp's 32 rows are contiguous in global memory (32 x 3K floats),
// so they are loaded and stored with fully coalesced 128-bit accesses by flat position, and each thread
// reads / writes its own row in shared memory (row stride chosen so that 128-bit shared accesses of 8
// consecutive lanes cover all banks).  Rows of culled Gaussians are not read; their gradients are zeros.
template <int D>
struct ShRowLayout {
  static constexpr int K = (D + 1) * (D + 1);
  static constexpr int RK = 3 * K;                  // floats per row
  static constexpr bool VEC = (RK % 4) == 0;        // D = 1, 3
  static constexpr int STRIDE = VEC ? (((RK / 4) % 2) ? RK : RK + 4) : ((RK % 2) ? RK : RK + 1);
};

#ifndef PB_H
#define PB_H float
#endif

// Tail of the reverse pass, from dL/dU on.  Given dL/dU the remaining chain is sums of products of
// well-conditioned quantities, so it runs in H (fp32 by default; -DPB_H=double to compare).
struct GeoGrads {
  float dls[3];
  float4 dq;
  float dm[3];
};

template <typename H>
__device__ __forceinline__ GeoGrads geometry_tail(const H* Rd, bool xcl, bool ycl, H dU00, H dU01, H dU02, H dU10, H dU11, H dU12, H M00, H M01, H M02, H M10, H M11, H M12, H M20, H M21, H M22, H T00, H T01, H T02, H T10, H T11, H T12, H r00, H r01, H r02, H r10, H r11, H r12, H r20, H r21, H r22, H s0, H s1, H s2, H qw, H qx, H qy, H qz, H qinv, H fxd, H fyd, H iz, H tx, H ty, H xz, H yz, H gmx, H gmy, H dmx, H dmy, H dmz) {
  GeoGrads out;
  // U = T M:  dT = dU M^T,  dM = T^T dU
  const H dT00 = dU00 * M00 + dU01 * M01 + dU02 * M02, dT01 = dU00 * M10 + dU01 * M11 + dU02 * M12, dT02 = dU00 * M20 + dU01 * M21 + dU02 * M22;
  const H dT10 = dU10 * M00 + dU11 * M01 + dU12 * M02, dT11 = dU10 * M10 + dU11 * M11 + dU12 * M12, dT12 = dU10 * M20 + dU11 * M21 + dU12 * M22;
  const H dM00 = T00 * dU00 + T10 * dU10, dM01 = T00 * dU01 + T10 * dU11, dM02 = T00 * dU02 + T10 * dU12;
  const H dM10 = T01 * dU00 + T11 * dU10, dM11 = T01 * dU01 + T11 * dU11, dM12 = T01 * dU02 + T11 * dU12;
  const H dM20 = T02 * dU00 + T12 * dU10, dM21 = T02 * dU01 + T12 * dU11, dM22 = T02 * dU02 + T12 * dU12;
  // M = Rot diag(s)
  const H ds0 = dM00 * r00 + dM10 * r10 + dM20 * r20;
  const H ds1 = dM01 * r01 + dM11 * r11 + dM21 * r21;
  const H ds2 = dM02 * r02 + dM12 * r12 + dM22 * r22;
  out.dls[0] = (float)(ds0 * s0);
  out.dls[1] = (float)(ds1 * s1);
  out.dls[2] = (float)(ds2 * s2);
  const H dr00 = dM00 * s0, dr01 = dM01 * s1, dr02 = dM02 * s2;
  const H dr10 = dM10 * s0, dr11 = dM11 * s1, dr12 = dM12 * s2;
  const H dr20 = dM20 * s0, dr21 = dM21 * s1, dr22 = dM22 * s2;
  // Rot(unit quaternion)
  const H dqw = (H)2. * (-qz * dr01 + qy * dr02 + qz * dr10 - qx * dr12 - qy * dr20 + qx * dr21);
  const H dqx = (H)2. * (qy * dr01 + qz * dr02 + qy * dr10 - (H)2. * qx * dr11 - qw * dr12 + qz * dr20 + qw * dr21 - (H)2. * qx * dr22);
  const H dqy = (H)2. * (-(H)2. * qy * dr00 + qx * dr01 + qw * dr02 + qx * dr10 + qz * dr12 - qw * dr20 + qz * dr21 - (H)2. * qy * dr22);
  const H dqz = (H)2. * (-(H)2. * qz * dr00 - qw * dr01 + qx * dr02 + qw * dr10 - (H)2. * qz * dr11 + qy * dr12 + qx * dr20 + qy * dr21);
  // through q / |q|
  const H qdot = qw * dqw + qx * dqx + qy * dqy + qz * dqz;
  out.dq = make_float4((float)((dqw - qw * qdot) * qinv), (float)((dqx - qx * qdot) * qinv), (float)((dqy - qy * qdot) * qinv), (float)((dqz - qz * qdot) * qinv));
  // T = J W
  const H dJ00 = dT00 * Rd[0] + dT01 * Rd[1] + dT02 * Rd[2];
  const H dJ02 = dT00 * Rd[6] + dT01 * Rd[7] + dT02 * Rd[8];
  const H dJ11 = dT10 * Rd[3] + dT11 * Rd[4] + dT12 * Rd[5];
  const H dJ12 = dT10 * Rd[6] + dT11 * Rd[7] + dT12 * Rd[8];
  // J(t) and the projected centre
  const H iz2 = iz * iz;
  H dtx = gmx * fxd * iz, dty = gmy * fyd * iz;
  H dtz = -(dJ00 * fxd + dJ11 * fyd) * iz2 - ((H)gmx * fxd * tx + (H)gmy * fyd * ty) * iz2;
  if (xcl) dtz += dJ02 * fxd * xz * iz2;  // J02 = -fx L / z with L = +-limx
  else { dtx += -dJ02 * fxd * iz2; dtz += dJ02 * (H)2. * fxd * tx * iz2 * iz; }
  if (ycl) dtz += dJ12 * fyd * yz * iz2;
  else { dty += -dJ12 * fyd * iz2; dtz += dJ12 * (H)2. * fyd * ty * iz2 * iz; }
  // t = R p + t_cam
  const H dmx_g = Rd[0] * dtx + Rd[3] * dty + Rd[6] * dtz;
  const H dmy_g = Rd[1] * dtx + Rd[4] * dty + Rd[7] * dtz;
  const H dmz_g = Rd[2] * dtx + Rd[5] * dty + Rd[8] * dtz;
  out.dm[0] = (float)((H)dmx + dmx_g);
  out.dm[1] = (float)((H)dmy + dmy_g);
  out.dm[2] = (float)((H)dmz + dmz_g);
  return out;
}

constexpr int PB_THREADS = 128;
#ifndef PB_G
#define PB_G double
#endif

// Kernel 1 of 2: colour.  dL/dsh, and the part of dL/dmean that flows through the view direction (written to
// dL_dmeans; kernel 2 adds the geometric part).  fp32, light on registers, HBM-bound.
template <int D>
__global__ void __launch_bounds__(PB_THREADS) preprocess_bwd_sh_kernel(
    mg_camera cam, int64_t N, const float* __restrict__ means, const float* __restrict__ sh,
    const int32_t* __restrict__ radii, const uint8_t* __restrict__ clamped, const float* __restrict__ dL_drgb,
    float* __restrict__ dL_dmeans, float* __restrict__ dL_dsh) {
  typedef ShRowLayout<D> L;
  constexpr int K = L::K, RK = L::RK, STRIDE = L::STRIDE;
  __shared__ __align__(16) float rows_all[PB_THREADS / 32][32 * STRIDE];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  float* wrow = rows_all[warp];
  float* myrow = wrow + lane * STRIDE;
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int64_t g0 = i - lane;                              // first Gaussian of this warp
  const int nrows = (int)max((int64_t)0, min((int64_t)32, N - g0));
  // A Gaussian whose colour received no gradient (culled, every channel clamped, or -- the common case -- never
  // reached by a pixel before the pixel saturated) has dL/dsh = 0 and no direction term: its row is not read.
  // (every small load is issued before any is tested: dependent loads would serialise their latencies)
  const bool in = i < N;
  const int rad = in ? radii[i] : 0;
  const uint32_t cl = in ? clamped[i] : 7u;
  float gcol[3];
#pragma unroll
  for (int k = 0; k < 3; k++) gcol[k] = in ? dL_drgb[3 * i + k] : 0.f;
  const float px = in ? means[3 * i] : 0.f, py = in ? means[3 * i + 1] : 0.f, pz = in ? means[3 * i + 2] : 0.f;
#pragma unroll
  for (int k = 0; k < 3; k++)
    if (cl >> k & 1u) gcol[k] = 0.f;
  const bool vis = rad > 0 && ((gcol[0] != 0.f) | (gcol[1] != 0.f) | (gcol[2] != 0.f));
  const uint32_t vmask = __ballot_sync(0xffffffffu, vis);
  // coalesced load of the visible rows
  if (nrows > 0) {
    if constexpr (L::VEC) {
      // asynchronous copies, all of a lane's in flight at once (see mg_preprocess)
      const float4* src = reinterpret_cast<const float4*>(sh + g0 * RK);
#pragma unroll
      for (int k = 0; k < RK / 4; k++) {
        const int f = k * 32 + lane, g = f / (RK / 4), c = f % (RK / 4);
        if (g < nrows && ((vmask >> g) & 1u)) mg_cp_async16(wrow + g * STRIDE + 4 * c, src + f);
      }
      mg_cp_async_commit();
      mg_cp_async_wait_all();
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
  if (vis) {
  const float* R = cam.R;
  // ---------------- colour: dL/dsh and the direction-dependent part of dL/dmean ----------------
  const float cpx = -(R[0] * cam.t[0] + R[3] * cam.t[1] + R[6] * cam.t[2]);
  const float cpy = -(R[1] * cam.t[0] + R[4] * cam.t[1] + R[7] * cam.t[2]);
  const float cpz = -(R[2] * cam.t[0] + R[5] * cam.t[1] + R[8] * cam.t[2]);
  const float vx = px - cpx, vy = py - cpy, vz = pz - cpz;
  const float ninv = rsqrtf(vx * vx + vy * vy + vz * vz);
  const float x = vx * ninv, y = vy * ninv, z = vz * ninv;
  float dmx = 0.f, dmy = 0.f, dmz = 0.f;  // dL/dmean (world)
  {
    // s_j = sum_k gcol_k sh[j][k];  dL/dsh[j][k] = Y_j gcol_k
    float sj[K], Y[K];
    {
      float rowv[RK];
      if constexpr (L::VEC) {
#pragma unroll
        for (int j = 0; j < RK / 4; j++) {
          const float4 v = *reinterpret_cast<const float4*>(myrow + 4 * j);
          rowv[4 * j] = v.x; rowv[4 * j + 1] = v.y; rowv[4 * j + 2] = v.z; rowv[4 * j + 3] = v.w;
        }
      } else {
#pragma unroll
        for (int j = 0; j < RK; j++) rowv[j] = myrow[j];
      }
#pragma unroll
      for (int j = 0; j < K; j++) sj[j] = gcol[0] * rowv[3 * j] + gcol[1] * rowv[3 * j + 1] + gcol[2] * rowv[3 * j + 2];
    }
    const float xx = x * x, yy = y * y, zz = z * z;
    Y[0] = MG_SH_C0;
    float ddx = 0.f, ddy = 0.f, ddz = 0.f;  // dL/d(direction) treating Y_j as polynomials on R^3
    if (D >= 1) {
      Y[1] = -MG_SH_C1 * y; Y[2] = MG_SH_C1 * z; Y[3] = -MG_SH_C1 * x;
      ddy += -MG_SH_C1 * sj[1];
      ddz += MG_SH_C1 * sj[2];
      ddx += -MG_SH_C1 * sj[3];
    }
    if (D >= 2) {
      Y[4] = MG_SH_C2_0 * (x * y); Y[5] = MG_SH_C2_1 * (y * z); Y[6] = MG_SH_C2_2 * (2.f * zz - xx - yy);
      Y[7] = MG_SH_C2_3 * (x * z); Y[8] = MG_SH_C2_4 * (xx - yy);
      ddx += MG_SH_C2_0 * y * sj[4] + MG_SH_C2_2 * (-2.f * x) * sj[6] + MG_SH_C2_3 * z * sj[7] + MG_SH_C2_4 * (2.f * x) * sj[8];
      ddy += MG_SH_C2_0 * x * sj[4] + MG_SH_C2_1 * z * sj[5] + MG_SH_C2_2 * (-2.f * y) * sj[6] + MG_SH_C2_4 * (-2.f * y) * sj[8];
      ddz += MG_SH_C2_1 * y * sj[5] + MG_SH_C2_2 * (4.f * z) * sj[6] + MG_SH_C2_3 * x * sj[7];
    }
    if (D >= 3) {
      Y[9] = MG_SH_C3_0 * (y * (3.f * xx - yy)); Y[10] = MG_SH_C3_1 * (x * y * z);
      Y[11] = MG_SH_C3_2 * (y * (4.f * zz - xx - yy)); Y[12] = MG_SH_C3_3 * (z * (2.f * zz - 3.f * xx - 3.f * yy));
      Y[13] = MG_SH_C3_4 * (x * (4.f * zz - xx - yy)); Y[14] = MG_SH_C3_5 * (z * (xx - yy));
      Y[15] = MG_SH_C3_6 * (x * (xx - 3.f * yy));
      ddx += MG_SH_C3_0 * (6.f * x * y) * sj[9] + MG_SH_C3_1 * (y * z) * sj[10] + MG_SH_C3_2 * (-2.f * x * y) * sj[11] +
             MG_SH_C3_3 * (-6.f * x * z) * sj[12] + MG_SH_C3_4 * (4.f * zz - 3.f * xx - yy) * sj[13] +
             MG_SH_C3_5 * (2.f * x * z) * sj[14] + MG_SH_C3_6 * (3.f * xx - 3.f * yy) * sj[15];
      ddy += MG_SH_C3_0 * (3.f * xx - 3.f * yy) * sj[9] + MG_SH_C3_1 * (x * z) * sj[10] +
             MG_SH_C3_2 * (4.f * zz - xx - 3.f * yy) * sj[11] + MG_SH_C3_3 * (-6.f * y * z) * sj[12] +
             MG_SH_C3_4 * (-2.f * x * y) * sj[13] + MG_SH_C3_5 * (-2.f * y * z) * sj[14] + MG_SH_C3_6 * (-6.f * x * y) * sj[15];
      ddz += MG_SH_C3_1 * (x * y) * sj[10] + MG_SH_C3_2 * (8.f * y * z) * sj[11] +
             MG_SH_C3_3 * (6.f * zz - 3.f * xx - 3.f * yy) * sj[12] + MG_SH_C3_4 * (8.f * x * z) * sj[13] +
             MG_SH_C3_5 * (xx - yy) * sj[14];
    }
    // through the normalisation d = v / |v|
    const float dot = x * ddx + y * ddy + z * ddz;
    dmx = (ddx - x * dot) * ninv;
    dmy = (ddy - y * dot) * ninv;
    dmz = (ddz - z * dot) * ninv;
    float out[3 * K];
#pragma unroll
    for (int j = 0; j < K; j++) {
      out[3 * j] = Y[j] * gcol[0]; out[3 * j + 1] = Y[j] * gcol[1]; out[3 * j + 2] = Y[j] * gcol[2];
    }
    if constexpr (L::VEC) {
#pragma unroll
      for (int j = 0; j < RK / 4; j++)
        *reinterpret_cast<float4*>(myrow + 4 * j) = make_float4(out[4 * j], out[4 * j + 1], out[4 * j + 2], out[4 * j + 3]);
    } else {
#pragma unroll
      for (int j = 0; j < RK; j++) myrow[j] = out[j];
    }
  }

    dL_dmeans[3 * i] = dmx; dL_dmeans[3 * i + 1] = dmy; dL_dmeans[3 * i + 2] = dmz;
  } else if (i < N) {
    dL_dmeans[3 * i] = dL_dmeans[3 * i + 1] = dL_dmeans[3 * i + 2] = 0.f;
  }
  __syncwarp();
  // coalesced store of dL/dsh: rows of visible Gaussians from shared memory, zeros for the others
  if (nrows > 0) {
    if constexpr (L::VEC) {
      float4* dst = reinterpret_cast<float4*>(dL_dsh + g0 * RK);
#pragma unroll
      for (int k = 0; k < RK / 4; k++) {
        const int f = k * 32 + lane, g = f / (RK / 4), c = f % (RK / 4);
        if (g < nrows) {
          float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
          if ((vmask >> g) & 1u) v = *reinterpret_cast<const float4*>(wrow + g * STRIDE + 4 * c);
          dst[f] = v;
        }
      }
    } else {
      float* dst = dL_dsh + g0 * RK;
#pragma unroll
      for (int k = 0; k < RK; k++) {
        const int f = k * 32 + lane, g = f / RK, c = f % RK;
        if (g < nrows) dst[f] = ((vmask >> g) & 1u) ? wrow[g * STRIDE + c] : 0.f;
      }
    }
  }
}


// Kernel 2 of 2: geometry.  Adds its part to dL_dmeans (written by kernel 1) and writes the other gradients.
// The chain of one Gaussian:
__device__ __forceinline__ void geo_one(const mg_camera& cam, int64_t i, const float* __restrict__ means,
                                        const float* __restrict__ log_scales, const float* __restrict__ quats,
                                        const float* __restrict__ opacity_logits, const float2* __restrict__ dL_dmeans2d,
                                        const float* __restrict__ dL_dconic, const float* __restrict__ dL_dopacity,
                                        float* __restrict__ dL_dmeans, float* __restrict__ dL_dlog_scales,
                                        float4* __restrict__ dL_dquats, float* __restrict__ dL_dopacity_logits) {
  const float2 gm = dL_dmeans2d[i];
  const float gA = dL_dconic[3 * i], gB = dL_dconic[3 * i + 1], gC = dL_dconic[3 * i + 2];
  const float go = dL_dopacity[i];
  const float px = means[3 * i], py = means[3 * i + 1], pz = means[3 * i + 2];
  const float4 q = __ldg(reinterpret_cast<const float4*>(quats) + i);
  const double s0 = exp((double)log_scales[3 * i]), s1 = exp((double)log_scales[3 * i + 1]), s2 = exp((double)log_scales[3 * i + 2]);
  const float o = 1.f / (1.f + expf(-opacity_logits[i]));
  const float dmx = dL_dmeans[3 * i], dmy = dL_dmeans[3 * i + 1], dmz = dL_dmeans[3 * i + 2];  // colour part

  // ---------------- geometry: forward chain and dL/dconic -> dL/dU in fp64 ----------------
  // dL/dconic is a sum of q d d^T over pixels; mapping it back through conic = Sigma2D^-1 contracts it
  // with vectors (A,B).d that are small for d along the major axis of an elongated splat, so the three
  // products cancel to ~(k2/k1)^2 of their size.  fp32 loses up to 1e-3 of dL/dlog_scale there, so the
  // forward chain up to det and the step conic -> covariance -> U run in fp64 on the fp32 inputs
  // (~200 fp64 flops per Gaussian); the rest of the reverse pass is fp32.
  typedef PB_G G;
  G Rd[9], td[3];
#pragma unroll
  for (int j = 0; j < 9; j++) Rd[j] = (G)cam.R[j];
#pragma unroll
  for (int j = 0; j < 3; j++) td[j] = (G)cam.t[j];
  const G fxd = (G)cam.fx, fyd = (G)cam.fy;
  const G pxd = px, pyd = py, pzd = pz;
  const G tx = Rd[0] * pxd + Rd[1] * pyd + Rd[2] * pzd + td[0];
  const G ty = Rd[3] * pxd + Rd[4] * pyd + Rd[5] * pzd + td[1];
  const G tz = Rd[6] * pxd + Rd[7] * pyd + Rd[8] * pzd + td[2];
  const G qn2 = (G)q.x * q.x + (G)q.y * q.y + (G)q.z * q.z + (G)q.w * q.w;
  const G qinv = (G)1 / sqrt(qn2);
  const G qw = q.x * qinv, qx = q.y * qinv, qy = q.z * qinv, qz = q.w * qinv;
  const G r00 = (G)1. - (G)2. * (qy * qy + qz * qz), r01 = (G)2. * (qx * qy - qw * qz), r02 = (G)2. * (qx * qz + qw * qy);
  const G r10 = (G)2. * (qx * qy + qw * qz), r11 = (G)1. - (G)2. * (qx * qx + qz * qz), r12 = (G)2. * (qy * qz - qw * qx);
  const G r20 = (G)2. * (qx * qz - qw * qy), r21 = (G)2. * (qy * qz + qw * qx), r22 = (G)1. - (G)2. * (qx * qx + qy * qy);
  const G M00 = r00 * s0, M01 = r01 * s1, M02 = r02 * s2;
  const G M10 = r10 * s0, M11 = r11 * s1, M12 = r12 * s2;
  const G M20 = r20 * s0, M21 = r21 * s1, M22 = r22 * s2;
  const G limx = (G)MG_JCLAMP * cam.width / ((G)2. * fxd), limy = (G)MG_JCLAMP * cam.height / ((G)2. * fyd);
  const G iz = (G)1. / tz;
  const G xz_raw = tx * iz, yz_raw = ty * iz;
  const bool xcl = xz_raw < -limx || xz_raw > limx, ycl = yz_raw < -limy || yz_raw > limy;
  const G xz = fmin(limx, fmax(-limx, xz_raw)), yz = fmin(limy, fmax(-limy, yz_raw));
  const G J00 = fxd * iz, J02 = -fxd * xz * iz, J11 = fyd * iz, J12 = -fyd * yz * iz;
  const G T00 = J00 * Rd[0] + J02 * Rd[6], T01 = J00 * Rd[1] + J02 * Rd[7], T02 = J00 * Rd[2] + J02 * Rd[8];
  const G T10 = J11 * Rd[3] + J12 * Rd[6], T11 = J11 * Rd[4] + J12 * Rd[7], T12 = J11 * Rd[5] + J12 * Rd[8];
  const G U00 = T00 * M00 + T01 * M10 + T02 * M20, U01 = T00 * M01 + T01 * M11 + T02 * M21, U02 = T00 * M02 + T01 * M12 + T02 * M22;
  const G U10 = T10 * M00 + T11 * M10 + T12 * M20, U11 = T10 * M01 + T11 * M11 + T12 * M21, U12 = T10 * M02 + T11 * M12 + T12 * M22;
  const G n0 = U00 * U00 + U01 * U01 + U02 * U02, n1 = U10 * U10 + U11 * U11 + U12 * U12;
  const G a = n0 + (G)MG_DILATION;
  const G b = U00 * U10 + U01 * U11 + U02 * U12;
  const G c = n1 + (G)MG_DILATION;
  // det = a c - b^2 as a sum of non-negative terms (see preprocess.cu)
  const G crx = U01 * U12 - U02 * U11, cry = U02 * U10 - U00 * U12, crz = U00 * U11 - U01 * U10;
  const G det = (crx * crx + cry * cry + crz * crz) + (G)MG_DILATION * (n0 + n1) + (G)MG_DILATION * (G)MG_DILATION;
  const G idet = (G)1. / det, idet2 = idet * idet;

  // ---------------- reverse ----------------
  // conic (A,B,C) = (c,-b,a)/det  ->  covariance (a,b,c)
  const G da = idet2 * (-c * c * gA + b * c * gB - b * b * gC);
  const G db = idet2 * ((G)2. * b * c * gA - (a * c + b * b) * gB + (G)2. * a * b * gC);
  const G dc = idet2 * (-b * b * gA + a * b * gB - a * a * gC);
  // a = U0.U0, b = U0.U1, c = U1.U1
  const G dU00 = (G)2. * da * U00 + db * U10, dU01 = (G)2. * da * U01 + db * U11, dU02 = (G)2. * da * U02 + db * U12;
  const G dU10 = (G)2. * dc * U10 + db * U00, dU11 = (G)2. * dc * U11 + db * U01, dU12 = (G)2. * dc * U12 + db * U02;
  // from dL/dU on: well-conditioned, fp32 (see geometry_tail)
  typedef PB_H H;
  H Rh[9];
#pragma unroll
  for (int j = 0; j < 9; j++) Rh[j] = (H)cam.R[j];
  const GeoGrads gg = geometry_tail<H>(Rh, xcl, ycl, (H)dU00, (H)dU01, (H)dU02, (H)dU10, (H)dU11, (H)dU12, (H)M00, (H)M01, (H)M02, (H)M10, (H)M11, (H)M12, (H)M20, (H)M21, (H)M22, (H)T00, (H)T01, (H)T02, (H)T10, (H)T11, (H)T12, (H)r00, (H)r01, (H)r02, (H)r10, (H)r11, (H)r12, (H)r20, (H)r21, (H)r22, (H)s0, (H)s1, (H)s2, (H)qw, (H)qx, (H)qy, (H)qz, (H)qinv, (H)fxd, (H)fyd, (H)iz, (H)tx, (H)ty, (H)xz, (H)yz, (H)gm.x, (H)gm.y, (H)dmx, (H)dmy, (H)dmz);
  dL_dlog_scales[3 * i] = gg.dls[0]; dL_dlog_scales[3 * i + 1] = gg.dls[1]; dL_dlog_scales[3 * i + 2] = gg.dls[2];
  dL_dquats[i] = gg.dq;
  dL_dmeans[3 * i] = gg.dm[0]; dL_dmeans[3 * i + 1] = gg.dm[1]; dL_dmeans[3 * i + 2] = gg.dm[2];
  dL_dopacity_logits[i] = go * o * ((G)1. - o);
}

// Only Gaussians that received a gradient need the chain, and once the pixels saturate few do (1 in 5 at config 3,
// scattered over the array), so the kernel is a persistent grid whose blocks sweep a contiguous range: a sweep
// step writes the zeros of 256 Gaussians that need none and appends the indices of the others to a queue in
// shared memory; whenever the queue holds 256 indices, all 8 warps run the fp64 chain on full lanes.
constexpr int PG_THREADS = 256;
constexpr int PG_SWEEP = 4;  // Gaussians per thread and sweep step

__global__ void __launch_bounds__(PG_THREADS, 2) preprocess_bwd_geo_kernel(
    mg_camera cam, int64_t N, const float* __restrict__ means, const float* __restrict__ log_scales,
    const float* __restrict__ quats, const float* __restrict__ opacity_logits, const int32_t* __restrict__ radii,
    const float2* __restrict__ dL_dmeans2d, const float* __restrict__ dL_dconic, const float* __restrict__ dL_dopacity,
    float* __restrict__ dL_dmeans, float* __restrict__ dL_dlog_scales, float4* __restrict__ dL_dquats,
    float* __restrict__ dL_dopacity_logits) {
  __shared__ uint32_t queue[(PG_SWEEP + 1) * PG_THREADS];  // indices relative to the block's range
  __shared__ uint32_t wcount[PG_THREADS / 32];
  __shared__ uint32_t qn;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  constexpr int STEP = PG_SWEEP * PG_THREADS;
  const int64_t per = ((N + gridDim.x - 1) / gridDim.x + STEP - 1) / STEP * STEP;
  const int64_t begin = (int64_t)blockIdx.x * per, end = min(N, begin + per);
  if (threadIdx.x == 0) qn = 0;
  __syncthreads();
  int64_t i0 = begin;
  for (;;) {
    // A sweep appends up to PG_SWEEP x 256 indices and a drain removes at most 256, so a sweep may only start while
    // fewer than 256 are queued: the queue then never holds more than 255 + PG_SWEEP x 256 < its capacity, whatever the
    // density of Gaussians with a gradient (qn is the same in every thread: it is only written in front of a barrier).
    if (i0 < end && qn < PG_THREADS) {
      // sweep PG_SWEEP x 256 Gaussians: all their loads are in flight together
      // every load is issued before any is tested (no short-circuit: dependent loads would serialise the latency)
      bool active[PG_SWEEP];
      int rad[PG_SWEEP];
      float2 gm_[PG_SWEEP];
      float gc_[PG_SWEEP][3], go_[PG_SWEEP];
#pragma unroll
      for (int u = 0; u < PG_SWEEP; u++) {
        const int64_t i = i0 + u * PG_THREADS + threadIdx.x;
        const bool in = i < end;
        rad[u] = in ? radii[i] : 0;
        gm_[u] = in ? dL_dmeans2d[i] : make_float2(0.f, 0.f);
        gc_[u][0] = in ? dL_dconic[3 * i] : 0.f;
        gc_[u][1] = in ? dL_dconic[3 * i + 1] : 0.f;
        gc_[u][2] = in ? dL_dconic[3 * i + 2] : 0.f;
        go_[u] = in ? dL_dopacity[i] : 0.f;
      }
#pragma unroll
      for (int u = 0; u < PG_SWEEP; u++)
        active[u] = rad[u] > 0 && ((gm_[u].x != 0.f) | (gm_[u].y != 0.f) | (gc_[u][0] != 0.f) | (gc_[u][1] != 0.f) |
                                   (gc_[u][2] != 0.f) | (go_[u] != 0.f));
#pragma unroll
      for (int u = 0; u < PG_SWEEP; u++) {
        const int64_t i = i0 + u * PG_THREADS + threadIdx.x;
        if (i < end && !active[u]) {
          // culled, or no gradient reached this Gaussian (no pixel blended it before saturating): exact zeros
          // (dL_dmeans holds the colour part, zero as well, from kernel 1)
          dL_dlog_scales[3 * i] = dL_dlog_scales[3 * i + 1] = dL_dlog_scales[3 * i + 2] = 0.f;
          dL_dquats[i] = make_float4(0.f, 0.f, 0.f, 0.f);
          dL_dopacity_logits[i] = 0.f;
        }
        const uint32_t ballot = __ballot_sync(0xffffffffu, active[u]);
        if (lane == 0) wcount[warp] = __popc(ballot);
        __syncthreads();
        uint32_t off = qn, tot = 0;
#pragma unroll
        for (int w = 0; w < PG_THREADS / 32; w++) {
          if (w < warp) off += wcount[w];
          tot += wcount[w];
        }
        if (active[u]) queue[off + __popc(ballot & ((1u << lane) - 1u))] = (uint32_t)(i - begin);
        __syncthreads();
        if (threadIdx.x == 0) qn += tot;
        __syncthreads();
      }
      i0 += STEP;
    }
    const uint32_t n = qn;  // same value in every thread
    const bool flush = i0 >= end;
    if (n >= PG_THREADS || (flush && n > 0)) {
      // run the chain on the LAST min(n, 256) entries of the queue: nothing to move afterwards
      const uint32_t cnt = min(n, (uint32_t)PG_THREADS);
      if (threadIdx.x < cnt)
        geo_one(cam, begin + queue[n - cnt + threadIdx.x], means, log_scales, quats, opacity_logits, dL_dmeans2d, dL_dconic,
                dL_dopacity, dL_dmeans, dL_dlog_scales, dL_dquats, dL_dopacity_logits);
      __syncthreads();
      if (threadIdx.x == 0) qn = n - cnt;
      __syncthreads();
    } else if (flush) {
      break;
    }
  }
}

}  // namespace

extern "C" int mg_preprocess_bwd(const mg_camera* cam, int64_t N, const float* means, const float* log_scales,
                                 const float* quats, const float* opacity_logits, const float* sh, const int32_t* radii,
                                 const uint8_t* clamped, const float* dL_dmeans2d, const float* dL_dconic,
                                 const float* dL_dopacity, const float* dL_drgb, float* dL_dmeans,
                                 float* dL_dlog_scales, float* dL_dquats, float* dL_dopacity_logits, float* dL_dsh,
                                 void* stream) {
  if (int rc = mg_check_camera(cam)) return rc;
  MG_REQUIRE(N >= 0 && N < (int64_t)1 << 31, "N must be in [0, 2^31)");
  if (N == 0) return MG_OK;
  MG_REQUIRE(means && log_scales && quats && opacity_logits && sh && radii && clamped, "null input array");
  MG_REQUIRE(dL_dmeans2d && dL_dconic && dL_dopacity && dL_drgb, "null upstream gradient");
  MG_REQUIRE(dL_dmeans && dL_dlog_scales && dL_dquats && dL_dopacity_logits && dL_dsh, "null output gradient");
  const int threads = PB_THREADS;
  const unsigned blocks = (unsigned)((N + threads - 1) / threads);
  cudaStream_t st = (cudaStream_t)stream;
#define MG_LAUNCH(D)                                                                                            \
  preprocess_bwd_sh_kernel<D><<<blocks, threads, 0, st>>>(*cam, N, means, sh, radii, clamped, dL_drgb, dL_dmeans, dL_dsh)
  switch (cam->sh_degree) {
    case 0: MG_LAUNCH(0); break;
    case 1: MG_LAUNCH(1); break;
    case 2: MG_LAUNCH(2); break;
    default: MG_LAUNCH(3); break;
  }
#undef MG_LAUNCH
  MG_CHECK_LAUNCH();
  int sms = 0;
  if (int rc = mg_current_device(nullptr, &sms)) return rc;
  const int geo_grid = 2 * sms;  // persistent grid: 2 blocks per SM
  const int64_t geo_want = (N + PG_THREADS - 1) / PG_THREADS;
  preprocess_bwd_geo_kernel<<<(unsigned)(geo_want < geo_grid ? geo_want : geo_grid), PG_THREADS, 0, st>>>(*cam, N, means, log_scales, quats, opacity_logits, radii,
                                                        (const float2*)dL_dmeans2d, dL_dconic, dL_dopacity, dL_dmeans,
                                                        dL_dlog_scales, (float4*)dL_dquats, dL_dopacity_logits);
  MG_CHECK_LAUNCH();
  return MG_OK;
}
