// preprocess_bwd.cu -- mg_preprocess_bwd: vector-Jacobian product of mg_preprocess (step a9).
// The paper gives no formulas for this step ("We modify the CUDA rasterization code of 3DGS",
// PAPER.md:156); it is the chain rule of DESIGN.md O1-O8, hand-derived here in reverse mode.  The
// oracle obtains the same quantity by forward-mode dual numbers, so the two derivations are independent.
// HBM-bound: one thread per Gaussian; 236 B of inputs + 36 B of upstream gradients in, 236 B out.
#include "mg_common.cuh"

namespace {

template <int D>
__global__ void __launch_bounds__(128) preprocess_bwd_kernel(
    mg_camera cam, int64_t N, const float* __restrict__ means, const float* __restrict__ log_scales,
    const float* __restrict__ quats, const float* __restrict__ opacity_logits, const float* __restrict__ sh,
    const int32_t* __restrict__ radii, const uint8_t* __restrict__ clamped, const float2* __restrict__ dL_dmeans2d,
    const float* __restrict__ dL_dconic, const float* __restrict__ dL_dopacity, const float* __restrict__ dL_drgb,
    float* __restrict__ dL_dmeans, float* __restrict__ dL_dlog_scales, float4* __restrict__ dL_dquats,
    float* __restrict__ dL_dopacity_logits, float* __restrict__ dL_dsh) {
  constexpr int K = (D + 1) * (D + 1);
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N) return;
  float* gsh = dL_dsh + i * (3 * K);
  if (radii[i] <= 0) {  // culled: exact zeros everywhere
    dL_dmeans[3 * i] = dL_dmeans[3 * i + 1] = dL_dmeans[3 * i + 2] = 0.f;
    dL_dlog_scales[3 * i] = dL_dlog_scales[3 * i + 1] = dL_dlog_scales[3 * i + 2] = 0.f;
    dL_dquats[i] = make_float4(0.f, 0.f, 0.f, 0.f);
    dL_dopacity_logits[i] = 0.f;
    if ((3 * K) % 4 == 0) {
#pragma unroll
      for (int j = 0; j < 3 * K / 4; j++) reinterpret_cast<float4*>(gsh)[j] = make_float4(0.f, 0.f, 0.f, 0.f);
    } else {
#pragma unroll
      for (int j = 0; j < 3 * K; j++) gsh[j] = 0.f;
    }
    return;
  }
  const float* R = cam.R;
  const float px = means[3 * i], py = means[3 * i + 1], pz = means[3 * i + 2];
  const float4 q = __ldg(reinterpret_cast<const float4*>(quats) + i);
  const float s0 = expf(log_scales[3 * i]), s1 = expf(log_scales[3 * i + 1]), s2 = expf(log_scales[3 * i + 2]);
  const float o = 1.f / (1.f + expf(-opacity_logits[i]));
  const float2 gm = dL_dmeans2d[i];
  const float gA = dL_dconic[3 * i], gB = dL_dconic[3 * i + 1], gC = dL_dconic[3 * i + 2];
  const uint32_t cl = clamped[i];
  float gcol[3];
#pragma unroll
  for (int k = 0; k < 3; k++) gcol[k] = (cl >> k & 1u) ? 0.f : dL_drgb[3 * i + k];

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
    const float* shrow = sh + i * (3 * K);
#pragma unroll
    for (int j = 0; j < K; j++)
      sj[j] = gcol[0] * __ldg(shrow + 3 * j) + gcol[1] * __ldg(shrow + 3 * j + 1) + gcol[2] * __ldg(shrow + 3 * j + 2);
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
    if ((3 * K) % 4 == 0) {
#pragma unroll
      for (int j = 0; j < 3 * K / 4; j++)
        reinterpret_cast<float4*>(gsh)[j] = make_float4(out[4 * j], out[4 * j + 1], out[4 * j + 2], out[4 * j + 3]);
    } else {
#pragma unroll
      for (int j = 0; j < 3 * K; j++) gsh[j] = out[j];
    }
  }

  // ---------------- geometry: recompute the forward quantities ----------------
  const float tx = R[0] * px + R[1] * py + R[2] * pz + cam.t[0];
  const float ty = R[3] * px + R[4] * py + R[5] * pz + cam.t[1];
  const float tz = R[6] * px + R[7] * py + R[8] * pz + cam.t[2];
  const float qn2 = q.x * q.x + q.y * q.y + q.z * q.z + q.w * q.w;
  const float qinv = rsqrtf(qn2);
  const float qw = q.x * qinv, qx = q.y * qinv, qy = q.z * qinv, qz = q.w * qinv;
  const float r00 = 1.f - 2.f * (qy * qy + qz * qz), r01 = 2.f * (qx * qy - qw * qz), r02 = 2.f * (qx * qz + qw * qy);
  const float r10 = 2.f * (qx * qy + qw * qz), r11 = 1.f - 2.f * (qx * qx + qz * qz), r12 = 2.f * (qy * qz - qw * qx);
  const float r20 = 2.f * (qx * qz - qw * qy), r21 = 2.f * (qy * qz + qw * qx), r22 = 1.f - 2.f * (qx * qx + qy * qy);
  const float M00 = r00 * s0, M01 = r01 * s1, M02 = r02 * s2;
  const float M10 = r10 * s0, M11 = r11 * s1, M12 = r12 * s2;
  const float M20 = r20 * s0, M21 = r21 * s1, M22 = r22 * s2;
  const float limx = MG_JCLAMP * cam.width / (2.f * cam.fx), limy = MG_JCLAMP * cam.height / (2.f * cam.fy);
  const float iz = 1.f / tz;
  const float xz_raw = tx * iz, yz_raw = ty * iz;
  const bool xcl = xz_raw < -limx || xz_raw > limx, ycl = yz_raw < -limy || yz_raw > limy;
  const float xz = fminf(limx, fmaxf(-limx, xz_raw)), yz = fminf(limy, fmaxf(-limy, yz_raw));
  const float J00 = cam.fx * iz, J02 = -cam.fx * xz * iz, J11 = cam.fy * iz, J12 = -cam.fy * yz * iz;
  const float T00 = J00 * R[0] + J02 * R[6], T01 = J00 * R[1] + J02 * R[7], T02 = J00 * R[2] + J02 * R[8];
  const float T10 = J11 * R[3] + J12 * R[6], T11 = J11 * R[4] + J12 * R[7], T12 = J11 * R[5] + J12 * R[8];
  const float U00 = T00 * M00 + T01 * M10 + T02 * M20, U01 = T00 * M01 + T01 * M11 + T02 * M21, U02 = T00 * M02 + T01 * M12 + T02 * M22;
  const float U10 = T10 * M00 + T11 * M10 + T12 * M20, U11 = T10 * M01 + T11 * M11 + T12 * M21, U12 = T10 * M02 + T11 * M12 + T12 * M22;
  const float a = U00 * U00 + U01 * U01 + U02 * U02 + MG_DILATION;
  const float b = U00 * U10 + U01 * U11 + U02 * U12;
  const float c = U10 * U10 + U11 * U11 + U12 * U12 + MG_DILATION;
  const float det = a * c - b * b;
  const float idet = 1.f / det, idet2 = idet * idet;

  // ---------------- reverse ----------------
  // conic (A,B,C) = (c,-b,a)/det  ->  covariance (a,b,c)
  const float da = idet2 * (-c * c * gA + b * c * gB - b * b * gC);
  const float db = idet2 * (2.f * b * c * gA - (a * c + b * b) * gB + 2.f * a * b * gC);
  const float dc = idet2 * (-b * b * gA + a * b * gB - a * a * gC);
  // a = U0.U0, b = U0.U1, c = U1.U1
  const float dU00 = 2.f * da * U00 + db * U10, dU01 = 2.f * da * U01 + db * U11, dU02 = 2.f * da * U02 + db * U12;
  const float dU10 = 2.f * dc * U10 + db * U00, dU11 = 2.f * dc * U11 + db * U01, dU12 = 2.f * dc * U12 + db * U02;
  // U = T M:  dT = dU M^T,  dM = T^T dU
  const float dT00 = dU00 * M00 + dU01 * M01 + dU02 * M02, dT01 = dU00 * M10 + dU01 * M11 + dU02 * M12, dT02 = dU00 * M20 + dU01 * M21 + dU02 * M22;
  const float dT10 = dU10 * M00 + dU11 * M01 + dU12 * M02, dT11 = dU10 * M10 + dU11 * M11 + dU12 * M12, dT12 = dU10 * M20 + dU11 * M21 + dU12 * M22;
  const float dM00 = T00 * dU00 + T10 * dU10, dM01 = T00 * dU01 + T10 * dU11, dM02 = T00 * dU02 + T10 * dU12;
  const float dM10 = T01 * dU00 + T11 * dU10, dM11 = T01 * dU01 + T11 * dU11, dM12 = T01 * dU02 + T11 * dU12;
  const float dM20 = T02 * dU00 + T12 * dU10, dM21 = T02 * dU01 + T12 * dU11, dM22 = T02 * dU02 + T12 * dU12;
  // M = Rot diag(s)
  const float ds0 = dM00 * r00 + dM10 * r10 + dM20 * r20;
  const float ds1 = dM01 * r01 + dM11 * r11 + dM21 * r21;
  const float ds2 = dM02 * r02 + dM12 * r12 + dM22 * r22;
  dL_dlog_scales[3 * i] = ds0 * s0;
  dL_dlog_scales[3 * i + 1] = ds1 * s1;
  dL_dlog_scales[3 * i + 2] = ds2 * s2;
  const float dr00 = dM00 * s0, dr01 = dM01 * s1, dr02 = dM02 * s2;
  const float dr10 = dM10 * s0, dr11 = dM11 * s1, dr12 = dM12 * s2;
  const float dr20 = dM20 * s0, dr21 = dM21 * s1, dr22 = dM22 * s2;
  // Rot(unit quaternion)
  const float dqw = 2.f * (-qz * dr01 + qy * dr02 + qz * dr10 - qx * dr12 - qy * dr20 + qx * dr21);
  const float dqx = 2.f * (qy * dr01 + qz * dr02 + qy * dr10 - 2.f * qx * dr11 - qw * dr12 + qz * dr20 + qw * dr21 - 2.f * qx * dr22);
  const float dqy = 2.f * (-2.f * qy * dr00 + qx * dr01 + qw * dr02 + qx * dr10 + qz * dr12 - qw * dr20 + qz * dr21 - 2.f * qy * dr22);
  const float dqz = 2.f * (-2.f * qz * dr00 - qw * dr01 + qx * dr02 + qw * dr10 - 2.f * qz * dr11 + qy * dr12 + qx * dr20 + qy * dr21);
  // through q / |q|
  const float qdot = qw * dqw + qx * dqx + qy * dqy + qz * dqz;
  dL_dquats[i] = make_float4((dqw - qw * qdot) * qinv, (dqx - qx * qdot) * qinv, (dqy - qy * qdot) * qinv, (dqz - qz * qdot) * qinv);
  // T = J W
  const float dJ00 = dT00 * R[0] + dT01 * R[1] + dT02 * R[2];
  const float dJ02 = dT00 * R[6] + dT01 * R[7] + dT02 * R[8];
  const float dJ11 = dT10 * R[3] + dT11 * R[4] + dT12 * R[5];
  const float dJ12 = dT10 * R[6] + dT11 * R[7] + dT12 * R[8];
  // J(t) and the projected centre
  const float iz2 = iz * iz;
  float dtx = gm.x * cam.fx * iz, dty = gm.y * cam.fy * iz;
  float dtz = -(dJ00 * cam.fx + dJ11 * cam.fy) * iz2 - (gm.x * cam.fx * tx + gm.y * cam.fy * ty) * iz2;
  if (xcl) dtz += dJ02 * cam.fx * xz * iz2;  // J02 = -fx L / z with L = +-limx
  else { dtx += -dJ02 * cam.fx * iz2; dtz += dJ02 * 2.f * cam.fx * tx * iz2 * iz; }
  if (ycl) dtz += dJ12 * cam.fy * yz * iz2;
  else { dty += -dJ12 * cam.fy * iz2; dtz += dJ12 * 2.f * cam.fy * ty * iz2 * iz; }
  // t = R p + t_cam
  dmx += R[0] * dtx + R[3] * dty + R[6] * dtz;
  dmy += R[1] * dtx + R[4] * dty + R[7] * dtz;
  dmz += R[2] * dtx + R[5] * dty + R[8] * dtz;
  dL_dmeans[3 * i] = dmx;
  dL_dmeans[3 * i + 1] = dmy;
  dL_dmeans[3 * i + 2] = dmz;
  dL_dopacity_logits[i] = dL_dopacity[i] * o * (1.f - o);
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
  const int threads = 128;
  const unsigned blocks = (unsigned)((N + threads - 1) / threads);
  cudaStream_t st = (cudaStream_t)stream;
#define MG_LAUNCH(D)                                                                                              \
  preprocess_bwd_kernel<D><<<blocks, threads, 0, st>>>(*cam, N, means, log_scales, quats, opacity_logits, sh,     \
                                                       radii, clamped, (const float2*)dL_dmeans2d, dL_dconic,     \
                                                       dL_dopacity, dL_drgb, dL_dmeans, dL_dlog_scales,           \
                                                       (float4*)dL_dquats, dL_dopacity_logits, dL_dsh)
  switch (cam->sh_degree) {
    case 0: MG_LAUNCH(0); break;
    case 1: MG_LAUNCH(1); break;
    case 2: MG_LAUNCH(2); break;
    default: MG_LAUNCH(3); break;
  }
#undef MG_LAUNCH
  MG_CHECK_LAUNCH();
  return MG_OK;
}
