// mg_oracle.cpp -- CPU ORACLE for the masked-rasterization hot path of MaskGaussian
// (arXiv 2412.20522; citations are /root/reference/PAPER.md line numbers + equation).
//
// THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
// bench.py's cpu_baseline / --impl reference legs may call it.  It shares no code, header,
// table or constant with paper_2412_20522_b200/csrc (the constants below are the oracle's own
// copy of the DESIGN.md readings).  Plain, slow, fp64; brute force in structure:
//   * per tile, the list is "every surviving Gaussian, in global depth order, whose tile
//     rectangle contains the tile" (no key sort, no binning structure);
//   * per pixel, the blend walks that list and applies Eq. 3-4 with the thresholds.
// OpenMP parallelises over Gaussians / tiles only (no blocking, fusion or reordering of the
// arithmetic).
//
// Steps (DESIGN.md "Oracle" O1..O12):
//   orc_preprocess      O1-O8   PAPER.md:64-66 (sec. 3.1), 74
//   orc_bin_sort        O9      PAPER.md:66 ("depth order"), 74 (16x16 tiles)
//   orc_render_fwd      O10     PAPER.md:86-90 (Eq. 3-4), 315-321 (Eq. 9-10)
//   orc_render_bwd      O11     PAPER.md:325 (Eq. 11), 336-364 (Eq. 13-18)
//   orc_preprocess_bwd  O12     chain rule of O1-O8, by forward-mode dual numbers through the
//                               SAME templated projection code (no hand-derived formulas)
//
// Parity pins: tests/test_oracle_pins.py (P1..P12).  "parity unpinned": the numeric values of
// the constants below and the SH sign convention (fixed by DESIGN.md, not by the paper).
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>

namespace {

// ---- the oracle's own copy of the readings (rows 1, 11-14) ----
const double ALPHA_MIN = 1.0 / 255.0;  // skip a pair when alpha < 1/255
const double ALPHA_MAX = 0.99;         // alpha = min(0.99, o*G)
const double T_MIN = 1e-4;             // stop when the post-blend T would fall below 1e-4
const int TILE = 16;
const double DILATION = 0.3;           // low-pass added to the 2D covariance diagonal
const double ZNEAR = 0.2;              // cull t.z <= 0.2
const double JCLAMP = 1.3;             // clamp x/z, y/z to +-1.3*tan(fov/2) inside J
const double EIG_FLOOR = 0.1;          // floor under the sqrt of the eigenvalue formula

struct Cam {
  int32_t width, height;
  double fx, fy, cx, cy;
  double R[9];
  double t[3];
  double bg[3];
  int32_t sh_degree;
};

// ---- forward-mode dual number: value + ND directional derivatives ----
template <int ND>
struct Dual {
  double v;
  double d[ND];
  Dual() : v(0) { for (int i = 0; i < ND; i++) d[i] = 0; }
  Dual(double x) : v(x) { for (int i = 0; i < ND; i++) d[i] = 0; }
};
template <int ND> Dual<ND> operator+(const Dual<ND>& a, const Dual<ND>& b) { Dual<ND> r; r.v = a.v + b.v; for (int i = 0; i < ND; i++) r.d[i] = a.d[i] + b.d[i]; return r; }
template <int ND> Dual<ND> operator-(const Dual<ND>& a, const Dual<ND>& b) { Dual<ND> r; r.v = a.v - b.v; for (int i = 0; i < ND; i++) r.d[i] = a.d[i] - b.d[i]; return r; }
template <int ND> Dual<ND> operator-(const Dual<ND>& a) { Dual<ND> r; r.v = -a.v; for (int i = 0; i < ND; i++) r.d[i] = -a.d[i]; return r; }
template <int ND> Dual<ND> operator*(const Dual<ND>& a, const Dual<ND>& b) { Dual<ND> r; r.v = a.v * b.v; for (int i = 0; i < ND; i++) r.d[i] = a.d[i] * b.v + a.v * b.d[i]; return r; }
template <int ND> Dual<ND> operator/(const Dual<ND>& a, const Dual<ND>& b) { Dual<ND> r; r.v = a.v / b.v; for (int i = 0; i < ND; i++) r.d[i] = (a.d[i] - r.v * b.d[i]) / b.v; return r; }
template <int ND> Dual<ND> operator+(const Dual<ND>& a, double b) { return a + Dual<ND>(b); }
template <int ND> Dual<ND> operator-(const Dual<ND>& a, double b) { return a - Dual<ND>(b); }
template <int ND> Dual<ND> operator*(const Dual<ND>& a, double b) { return a * Dual<ND>(b); }
template <int ND> Dual<ND> operator*(double a, const Dual<ND>& b) { return Dual<ND>(a) * b; }
template <int ND> Dual<ND> operator/(double a, const Dual<ND>& b) { return Dual<ND>(a) / b; }
template <int ND> Dual<ND> operator-(double a, const Dual<ND>& b) { return Dual<ND>(a) - b; }
template <int ND> Dual<ND> operator+(double a, const Dual<ND>& b) { return Dual<ND>(a) + b; }
template <int ND> Dual<ND> dexp(const Dual<ND>& a) { Dual<ND> r; r.v = std::exp(a.v); for (int i = 0; i < ND; i++) r.d[i] = r.v * a.d[i]; return r; }
template <int ND> Dual<ND> dsqrt(const Dual<ND>& a) { Dual<ND> r; r.v = std::sqrt(a.v); for (int i = 0; i < ND; i++) r.d[i] = a.d[i] / (2 * r.v); return r; }
inline double dexp(double a) { return std::exp(a); }
inline double dsqrt(double a) { return std::sqrt(a); }
inline double val(double a) { return a; }
template <int ND> double val(const Dual<ND>& a) { return a.v; }

// Everything orc_preprocess produces for one Gaussian.
template <class S>
struct Splat {
  bool culled;
  S m2x, m2y;       // projected centre, pixel-index coordinates (O6)
  S A, B, C;        // conic = inverse of the dilated 2D covariance (O5)
  S o;              // activated opacity (O1)
  S rgb[3];         // colour (O8)
  double depth;     // camera-space z (O2)
  int radius;       // ceil(3*sqrt(lambda_max)) (O7)
  int rect[4];      // x0,y0,x1,y1 in tile units, max exclusive (O7)
  unsigned clamped; // bit k: colour channel k clamped at 0
  double margin;    // smallest absolute distance of an integer/cull decision from its flip point
};

// Real SH basis, Condon-Shortley sign, order (l, m=-l..l), as polynomials of the unit vector
// (reading 16; PAPER.md:64 only says "spherical harmonics coefficients").
template <class S>
void sh_basis(int degree, const S& x, const S& y, const S& z, S* Y) {
  const double PI = 3.14159265358979323846;
  Y[0] = S(0.5 * std::sqrt(1.0 / PI));
  if (degree < 1) return;
  const double c1 = std::sqrt(3.0 / (4.0 * PI));
  Y[1] = -c1 * y;
  Y[2] = c1 * z;
  Y[3] = -c1 * x;
  if (degree < 2) return;
  S xx = x * x, yy = y * y, zz = z * z;
  Y[4] = (0.5 * std::sqrt(15.0 / PI)) * (x * y);
  Y[5] = (-0.5 * std::sqrt(15.0 / PI)) * (y * z);
  Y[6] = (0.25 * std::sqrt(5.0 / PI)) * (2.0 * zz - xx - yy);
  Y[7] = (-0.5 * std::sqrt(15.0 / PI)) * (x * z);
  Y[8] = (0.25 * std::sqrt(15.0 / PI)) * (xx - yy);
  if (degree < 3) return;
  Y[9] = (-0.25 * std::sqrt(35.0 / (2.0 * PI))) * (y * (3.0 * xx - yy));
  Y[10] = (0.5 * std::sqrt(105.0 / PI)) * (x * y * z);
  Y[11] = (-0.25 * std::sqrt(21.0 / (2.0 * PI))) * (y * (4.0 * zz - xx - yy));
  Y[12] = (0.25 * std::sqrt(7.0 / PI)) * (z * (2.0 * zz - 3.0 * xx - 3.0 * yy));
  Y[13] = (-0.25 * std::sqrt(21.0 / (2.0 * PI))) * (x * (4.0 * zz - xx - yy));
  Y[14] = (0.25 * std::sqrt(105.0 / PI)) * (z * (xx - yy));
  Y[15] = (-0.25 * std::sqrt(35.0 / (2.0 * PI))) * (x * (xx - 3.0 * yy));
}

inline double frac_dist(double q) { return std::fabs(q - std::round(q)); }

// O1-O8 for one Gaussian.  S = double (forward) or Dual (derivatives of the same code).
// p, ls, q, logit: the raw inputs; sh: K x 3 doubles.  Y_out (optional): SH basis values.
template <class S>
void project(const Cam& cam, const S p[3], const S ls[3], const S q[4], const S& logit,
             const double* sh, Splat<S>& out, double* Y_out) {
  const double* R = cam.R;
  out.culled = true;
  out.radius = 0;
  out.clamped = 0;
  out.margin = 1e30;
  out.rect[0] = out.rect[1] = out.rect[2] = out.rect[3] = 0;
  // O2 camera space (local affine transformation of ref [40])
  S tx = R[0] * p[0] + R[1] * p[1] + R[2] * p[2] + cam.t[0];
  S ty = R[3] * p[0] + R[4] * p[1] + R[5] * p[2] + cam.t[1];
  S tz = R[6] * p[0] + R[7] * p[1] + R[8] * p[2] + cam.t[2];
  out.depth = val(tz);
  out.margin = std::min(out.margin, std::fabs(val(tz) - ZNEAR));
  if (!(val(tz) > ZNEAR)) return;
  // O1 activations
  S s[3] = {dexp(ls[0]), dexp(ls[1]), dexp(ls[2])};
  S qn = dsqrt(q[0] * q[0] + q[1] * q[1] + q[2] * q[2] + q[3] * q[3]);
  S w = q[0] / qn, x = q[1] / qn, y = q[2] / qn, z = q[3] / qn;
  out.o = 1.0 / (1.0 + dexp(-logit));
  // O3 Sigma = Rot diag(s^2) Rot^T
  S Rot[9] = {1.0 - 2.0 * (y * y + z * z), 2.0 * (x * y - w * z),       2.0 * (x * z + w * y),
              2.0 * (x * y + w * z),       1.0 - 2.0 * (x * x + z * z), 2.0 * (y * z - w * x),
              2.0 * (x * z - w * y),       2.0 * (y * z + w * x),       1.0 - 2.0 * (x * x + y * y)};
  S M[9];
  for (int i = 0; i < 3; i++)
    for (int j = 0; j < 3; j++) M[3 * i + j] = Rot[3 * i + j] * s[j];
  S Sig[9];
  for (int i = 0; i < 3; i++)
    for (int j = 0; j < 3; j++) Sig[3 * i + j] = M[3 * i] * M[3 * j] + M[3 * i + 1] * M[3 * j + 1] + M[3 * i + 2] * M[3 * j + 2];
  // O4 Sigma2D = J W Sigma W^T J^T + 0.3 I, with the guard on x/z, y/z inside J only
  const double limx = JCLAMP * cam.width / (2.0 * cam.fx), limy = JCLAMP * cam.height / (2.0 * cam.fy);
  S xz = tx / tz, yz = ty / tz;
  if (val(xz) < -limx) xz = S(-limx); else if (val(xz) > limx) xz = S(limx);
  if (val(yz) < -limy) yz = S(-limy); else if (val(yz) > limy) yz = S(limy);
  S txc = xz * tz, tyc = yz * tz;
  S J00 = cam.fx / tz, J02 = -(cam.fx * txc) / (tz * tz);
  S J11 = cam.fy / tz, J12 = -(cam.fy * tyc) / (tz * tz);
  S T0[3], T1[3];
  for (int j = 0; j < 3; j++) {
    T0[j] = J00 * R[j] + J02 * R[6 + j];
    T1[j] = J11 * R[3 + j] + J12 * R[6 + j];
  }
  S u0[3], u1[3];  // Sigma * T0, Sigma * T1
  for (int i = 0; i < 3; i++) {
    u0[i] = Sig[3 * i] * T0[0] + Sig[3 * i + 1] * T0[1] + Sig[3 * i + 2] * T0[2];
    u1[i] = Sig[3 * i] * T1[0] + Sig[3 * i + 1] * T1[1] + Sig[3 * i + 2] * T1[2];
  }
  S a = T0[0] * u0[0] + T0[1] * u0[1] + T0[2] * u0[2] + DILATION;
  S b = T0[0] * u1[0] + T0[1] * u1[1] + T0[2] * u1[2];
  S c = T1[0] * u1[0] + T1[1] * u1[1] + T1[2] * u1[2] + DILATION;
  // O5 conic
  S det = a * c - b * b;
  if (!(val(det) > 0.0)) return;
  out.A = c / det;
  out.B = -b / det;
  out.C = a / det;
  // O6 projected centre; pixel (i,j) is evaluated at (i,j)
  out.m2x = cam.fx * tx / tz + (cam.cx - 0.5);
  out.m2y = cam.fy * ty / tz + (cam.cy - 0.5);
  // O7 radius and tile rectangle
  double mid = 0.5 * (val(a) + val(c));
  double lam = mid + std::sqrt(std::max(mid * mid - val(det), EIG_FLOOR));
  double r3 = 3.0 * std::sqrt(lam);
  int radius = (int)std::ceil(r3);
  out.margin = std::min(out.margin, frac_dist(r3));
  const int gw = (cam.width + TILE - 1) / TILE, gh = (cam.height + TILE - 1) / TILE;
  double qx0 = (val(out.m2x) - radius) / TILE, qx1 = (val(out.m2x) + radius + TILE - 1) / TILE;
  double qy0 = (val(out.m2y) - radius) / TILE, qy1 = (val(out.m2y) + radius + TILE - 1) / TILE;
  out.margin = std::min(out.margin, TILE * std::min(std::min(frac_dist(qx0), frac_dist(qx1)), std::min(frac_dist(qy0), frac_dist(qy1))));
  auto clampi = [](double v, int lo, int hi) { double f = std::floor(v); return f < lo ? lo : (f > hi ? hi : (int)f); };
  int x0 = clampi(qx0, 0, gw), x1 = clampi(qx1, 0, gw), y0 = clampi(qy0, 0, gh), y1 = clampi(qy1, 0, gh);
  if ((x1 - x0) * (y1 - y0) <= 0) return;
  out.radius = radius;
  out.rect[0] = x0; out.rect[1] = y0; out.rect[2] = x1; out.rect[3] = y1;
  // O8 colour from SH along the unit vector camera centre -> Gaussian centre
  double campos[3];
  for (int j = 0; j < 3; j++) campos[j] = -(R[j] * cam.t[0] + R[3 + j] * cam.t[1] + R[6 + j] * cam.t[2]);
  S dx = p[0] - campos[0], dy = p[1] - campos[1], dz = p[2] - campos[2];
  S dn = dsqrt(dx * dx + dy * dy + dz * dz);
  S Y[16];
  const int K = (cam.sh_degree + 1) * (cam.sh_degree + 1);
  sh_basis<S>(cam.sh_degree, dx / dn, dy / dn, dz / dn, Y);
  for (int k = 0; k < 3; k++) {
    S col(0.5);
    for (int j = 0; j < K; j++) col = col + Y[j] * sh[3 * j + k];
    if (val(col) < 0.0) { col = S(0.0); out.clamped |= 1u << k; }
    out.rgb[k] = col;
  }
  if (Y_out) for (int j = 0; j < K; j++) Y_out[j] = val(Y[j]);
  out.culled = false;
}

inline uint32_t float_bits(float f) { uint32_t u; std::memcpy(&u, &f, 4); return u; }

struct Passing {  // one list entry that passed the alpha filter at a pixel
  uint32_t pos;   // 1-based position in the tile list
  uint32_t id;
  double alpha, G, T, a, dx, dy;
  bool clamped;
};

}  // namespace

extern "C" {

// O1-O8.  Inputs are the caller's fp32 arrays upcast (exactly) to fp64 by the binding; the FD pin
// passes genuinely fp64 perturbed inputs.  Outputs are fp64 except the integers; culled Gaussians
// get zeros (radius 0).
int orc_preprocess(const Cam* cam, int64_t N, const double* means, const double* log_scales, const double* quats,
                   const double* opacity_logits, const double* sh, double* means2d, double* depths,
                   double* conic_opacity, double* rgb, int32_t* radii, int32_t* rects, uint32_t* tiles_touched,
                   uint8_t* clamped, double* margin) {
  const int K = (cam->sh_degree + 1) * (cam->sh_degree + 1);
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < N; i++) {
    double p[3], ls[3], q[4], shd[48];
    for (int j = 0; j < 3; j++) { p[j] = means[3 * i + j]; ls[j] = log_scales[3 * i + j]; }
    for (int j = 0; j < 4; j++) q[j] = quats[4 * i + j];
    for (int j = 0; j < 3 * K; j++) shd[j] = sh[(int64_t)3 * K * i + j];
    Splat<double> s;
    project<double>(*cam, p, ls, q, (double)opacity_logits[i], shd, s, nullptr);
    depths[i] = s.depth;
    margin[i] = s.margin;
    radii[i] = s.culled ? 0 : s.radius;
    for (int j = 0; j < 4; j++) rects[4 * i + j] = s.culled ? 0 : s.rect[j];
    tiles_touched[i] = s.culled ? 0u : (uint32_t)((s.rect[2] - s.rect[0]) * (s.rect[3] - s.rect[1]));
    clamped[i] = s.culled ? 0 : (uint8_t)s.clamped;
    means2d[2 * i] = s.culled ? 0 : s.m2x;
    means2d[2 * i + 1] = s.culled ? 0 : s.m2y;
    conic_opacity[4 * i + 0] = s.culled ? 0 : s.A;
    conic_opacity[4 * i + 1] = s.culled ? 0 : s.B;
    conic_opacity[4 * i + 2] = s.culled ? 0 : s.C;
    conic_opacity[4 * i + 3] = s.culled ? 0 : s.o;
    for (int k = 0; k < 3; k++) rgb[3 * i + k] = s.culled ? 0 : s.rgb[k];
  }
  return 0;
}

// O9.  Global order = surviving Gaussians ascending by the fp32 bit pattern of depth, ties by
// index (stable sort).  List of tile t = the sub-sequence of that order whose rect contains t.
// sorted_ids must hold R = sum(tiles_touched) entries; returns R through R_out.
// tile_select (optional, one byte per tile): tiles with a zero byte are left with an empty range, so
// that a bounded sample of a large workload can be listed (bench.py's cpu_baseline leg).
int orc_bin_sort(const Cam* cam, int64_t N, const float* depths, const int32_t* rects, const uint32_t* tiles_touched,
                 uint32_t* sorted_ids, uint32_t* tile_ranges, uint64_t* R_out, const uint8_t* tile_select) {
  const int gw = (cam->width + TILE - 1) / TILE, gh = (cam->height + TILE - 1) / TILE;
  std::vector<uint32_t> order;
  for (int64_t i = 0; i < N; i++)
    if (tiles_touched[i] > 0) order.push_back((uint32_t)i);
  std::stable_sort(order.begin(), order.end(), [&](uint32_t a, uint32_t b) { return float_bits(depths[a]) < float_bits(depths[b]); });
  const int ntiles = gw * gh;
  std::vector<uint64_t> count(ntiles + 1, 0);
#pragma omp parallel for schedule(dynamic, 4)
  for (int t = 0; t < ntiles; t++) {
    const int tx = t % gw, ty = t / gw;
    uint64_t c = 0;
    if (tile_select && !tile_select[t]) { count[t + 1] = 0; continue; }
    for (uint32_t id : order) {
      const int32_t* r = rects + 4 * (int64_t)id;
      if (tx >= r[0] && tx < r[2] && ty >= r[1] && ty < r[3]) c++;
    }
    count[t + 1] = c;
  }
  for (int t = 0; t < ntiles; t++) count[t + 1] += count[t];
#pragma omp parallel for schedule(dynamic, 4)
  for (int t = 0; t < ntiles; t++) {
    const int tx = t % gw, ty = t / gw;
    uint64_t k = count[t];
    if (!(tile_select && !tile_select[t]))
    for (uint32_t id : order) {
      const int32_t* r = rects + 4 * (int64_t)id;
      if (tx >= r[0] && tx < r[2] && ty >= r[1] && ty < r[3]) sorted_ids[k++] = id;
    }
    tile_ranges[2 * t] = (uint32_t)count[t];
    tile_ranges[2 * t + 1] = (uint32_t)count[t + 1];
  }
  *R_out = count[ntiles];
  return 0;
}

// Walk one pixel's list front to back (O10).  Fills `pass` (entries that passed the alpha
// filter and were blended) and returns the final transmittance.  `last` receives the number of list
// entries the pixel consumed: the entries in front of the one that stopped it, or the whole list if
// nothing stopped it (reading 5).  Every entry the reverse traversal must visit lies at a
// position <= last, and no entry at or behind the stop does.  `margin` receives the smallest
// relative distance of any decision from its flip point; `hash` a signature of all decisions.
// Work counters ("a pair evaluation = one (list entry, pixel) visited before the pixel stops; a
// blend = a pair evaluation that passes the alpha filter, masked or not"), split by the entry's mask:
//   cnt[0] / cnt[1]: entries visited with M != 0 / M == 0 (the entry that stops the pixel is visited: cnt[0]);
//   cnt[2] / cnt[3]: those of them that pass the alpha filter (the stopping entry passes it: cnt[2]).
static double walk_pixel(double px, double py, const uint32_t* ids, uint32_t n, const double* means2d,
                         const double* conic_opacity, const float* masks, std::vector<Passing>* pass, uint32_t* last,
                         double* margin, double* margin_clamp, uint64_t* hash, uint64_t* cnt) {
  double T = 1.0, mg = 1e30, mgc = 1e30;
  uint64_t h = 1469598103934665603ull;
  auto mix = [&](uint64_t v) { h = (h ^ v) * 1099511628211ull; };
  *last = n;
  for (uint32_t k = 0; k < n; k++) {
    const uint32_t id = ids[k];
    const int masked = masks[id] == 0.0f ? 1 : 0;
    cnt[masked]++;
    const double dx = means2d[2 * (int64_t)id] - px, dy = means2d[2 * (int64_t)id + 1] - py;
    const double* co = conic_opacity + 4 * (int64_t)id;
    const double power = -0.5 * (co[0] * dx * dx + 2.0 * co[1] * dx * dy + co[2] * dy * dy);
    if (power > 0.0) { mix(id * 4ull + 0); continue; }
    const double G = std::exp(power);
    const double oG = co[3] * G;
    const double alpha = std::min(ALPHA_MAX, oG);
    mg = std::min(mg, std::fabs(alpha - ALPHA_MIN) / ALPHA_MIN);
    if (alpha < ALPHA_MIN) { mix(id * 4ull + 1); continue; }  // the mask is NOT consulted
    cnt[2 + masked]++;
    mgc = std::min(mgc, std::fabs(oG - ALPHA_MAX) / ALPHA_MAX);
    const double a = (double)masks[id] * alpha;  // Eq. 4: T_{i+1} = (1 - M_i alpha_i) T_i
    const double Tn = T * (1.0 - a);
    mg = std::min(mg, std::fabs(Tn - T_MIN) / T_MIN);
    if (Tn < T_MIN) { mix(id * 4ull + 2); *last = k; break; }  // not blended, not counted: k entries consumed
    mix(id * 4ull + 3 + (oG > ALPHA_MAX ? 1ull << 40 : 0));
    if (pass) pass->push_back(Passing{k + 1, id, alpha, G, T, a, dx, dy, oG > ALPHA_MAX});
    T = Tn;
  }
  *margin = mg;
  *margin_clamp = mgc;
  *hash = h;
  return T;
}

// O10 forward: image = sum M_i c_i alpha_i T_i (Eq. 3) + T_{N+1} bg (Eq. 9-10).
// image [3][H][W], final_T [H][W], n_contrib [H][W] (number of list entries consumed before the stop,
// reading 5), margin [H][W], hash [H][W], counts[4] = walk_pixel's work counters summed over the pixels
// {pair evaluations M != 0, M == 0, blends M != 0, M == 0}.
int orc_render_fwd(const Cam* cam, const uint32_t* sorted_ids, const uint32_t* tile_ranges, const double* means2d,
                   const double* conic_opacity, const double* rgb, const float* masks, double* image, double* final_T,
                   uint32_t* n_contrib, double* margin, uint64_t* hash, uint64_t* counts) {
  const int W = cam->width, H = cam->height;
  const int gw = (W + TILE - 1) / TILE, gh = (H + TILE - 1) / TILE;
  uint64_t tot0 = 0, tot1 = 0, tot2 = 0, tot3 = 0;
#pragma omp parallel for schedule(dynamic, 1) reduction(+ : tot0, tot1, tot2, tot3)
  for (int t = 0; t < gw * gh; t++) {
    const uint32_t s = tile_ranges[2 * t], e = tile_ranges[2 * t + 1];
    std::vector<Passing> pass;
    for (int py = (t / gw) * TILE; py < std::min(H, (t / gw + 1) * TILE); py++)
      for (int px = (t % gw) * TILE; px < std::min(W, (t % gw + 1) * TILE); px++) {
        pass.clear();
        uint32_t last;
        double mg, mgc;
        uint64_t h, cnt[4] = {0, 0, 0, 0};
        const double T = walk_pixel(px, py, sorted_ids + s, e - s, means2d, conic_opacity, masks, &pass, &last, &mg, &mgc, &h, cnt);
        double C[3] = {0, 0, 0};
        for (const Passing& p : pass)
          for (int k = 0; k < 3; k++) C[k] += p.a * p.T * rgb[3 * (int64_t)p.id + k];
        const int64_t pix = (int64_t)py * W + px;
        for (int k = 0; k < 3; k++) image[(int64_t)k * H * W + pix] = C[k] + T * cam->bg[k];
        final_T[pix] = T;
        n_contrib[pix] = last;
        if (margin) margin[pix] = mg;
        if (hash) hash[pix] = h;
        tot0 += cnt[0]; tot1 += cnt[1]; tot2 += cnt[2]; tot3 += cnt[3];
      }
  }
  if (counts) { counts[0] = tot0; counts[1] = tot1; counts[2] = tot2; counts[3] = tot3; }
  return 0;
}

// O11 backward.  Per pixel: T_i from the forward walk (Eq. 13/16), b_{i+1} by the recursion of
// Eq. 11 from the back, then Eq. 18 for dL/dM_i; dL/dalpha_i = M_i * (same bracket); colour and
// alpha chain to (mean2d, conic, opacity).  All sums in fp64.
// sens[N] (optional): +1 for every pixel with a decision margin below `cutoff` at which the
// Gaussian was visited with alpha >= (1-cutoff)/255.  counts[4] = the work of the reverse traversal, which revisits
// positions n_contrib..1 of every pixel: {pair evaluations M != 0, M == 0, blends M != 0, M == 0} (the entry
// that stopped the pixel lies behind n_contrib and is not revisited).
int orc_render_bwd(const Cam* cam, int64_t N, const uint32_t* sorted_ids, const uint32_t* tile_ranges,
                   const double* means2d, const double* conic_opacity, const double* rgb, const float* masks,
                   const double* dL_dimage, double* dL_dmeans2d, double* dL_dconic, double* dL_dopacity,
                   double* dL_drgb, double* dL_dmask, uint32_t* sens, double cutoff, uint64_t* counts) {
  const int W = cam->width, H = cam->height;
  const int gw = (W + TILE - 1) / TILE, gh = (H + TILE - 1) / TILE;
  for (int64_t i = 0; i < N; i++) {
    dL_dmeans2d[2 * i] = dL_dmeans2d[2 * i + 1] = 0;
    dL_dconic[3 * i] = dL_dconic[3 * i + 1] = dL_dconic[3 * i + 2] = 0;
    dL_dopacity[i] = 0;
    dL_drgb[3 * i] = dL_drgb[3 * i + 1] = dL_drgb[3 * i + 2] = 0;
    dL_dmask[i] = 0;
    if (sens) sens[i] = 0;
  }
  uint64_t tot0 = 0, tot1 = 0, tot2 = 0, tot3 = 0;
#pragma omp parallel for schedule(dynamic, 1) reduction(+ : tot0, tot1, tot2, tot3)
  for (int t = 0; t < gw * gh; t++) {
    const uint32_t s = tile_ranges[2 * t], e = tile_ranges[2 * t + 1];
    const uint32_t n = e - s;
    if (n == 0) continue;
    std::vector<double> acc((size_t)n * 10, 0.0);  // per list entry: m2x,m2y,A,B,C,o,r,g,b,mask
    std::vector<uint32_t> sn(sens ? n : 0, 0);
    std::vector<Passing> pass;
    for (int py = (t / gw) * TILE; py < std::min(H, (t / gw + 1) * TILE); py++)
      for (int px = (t % gw) * TILE; px < std::min(W, (t % gw + 1) * TILE); px++) {
        pass.clear();
        uint32_t last;
        double mg, mgc;
        uint64_t h, cnt[4] = {0, 0, 0, 0};
        const double Tfin = walk_pixel(px, py, sorted_ids + s, n, means2d, conic_opacity, masks, &pass, &last, &mg, &mgc, &h, cnt);
        const uint64_t ne = cnt[0] + cnt[1];  // entries the forward walk visited (incl. the stopping one)
        const int64_t pix = (int64_t)py * W + px;
        const double g[3] = {dL_dimage[pix], dL_dimage[(int64_t)H * W + pix], dL_dimage[(int64_t)2 * H * W + pix]};
        const double gbg = g[0] * cam->bg[0] + g[1] * cam->bg[1] + g[2] * cam->bg[2];
        double Bc[3] = {0, 0, 0};  // b_{i+1}: colour rendered behind the current entry (Eq. 11), b_{N+1} = 0
        for (uint32_t k = 0; k < last; k++) {  // the reverse traversal revisits positions last..1
          if (masks[sorted_ids[s + k]] == 0.0f) tot1++; else tot0++;
        }
        for (const Passing& p : pass) {
          if (masks[p.id] == 0.0f) tot3++; else tot2++;
        }
        for (size_t kk = pass.size(); kk-- > 0;) {
          const Passing& p = pass[kk];
          const double* c = rgb + 3 * (int64_t)p.id;
          const double* co = conic_opacity + 4 * (int64_t)p.id;
          double* ac = acc.data() + (size_t)(p.pos - 1) * 10;
          // Eq. 18: alpha_i T_i g.(c_i - b_{i+1})  -  alpha_i T_{N+1}/(1 - alpha_i M_i) g.c_bg
          const double X = p.T * (g[0] * (c[0] - Bc[0]) + g[1] * (c[1] - Bc[1]) + g[2] * (c[2] - Bc[2])) - Tfin / (1.0 - p.a) * gbg;
          ac[9] += p.alpha * X;
          const double dalpha = (double)masks[p.id] * X;
          for (int k = 0; k < 3; k++) ac[6 + k] += p.a * p.T * g[k];
          for (int k = 0; k < 3; k++) Bc[k] = p.a * c[k] + (1.0 - p.a) * Bc[k];
          if (!p.clamped) {  // true derivative of min(0.99, o G): zero where the clamp is active
            ac[5] += p.G * dalpha;
            const double dpower = co[3] * p.G * dalpha;
            // power = -1/2 (A dx^2 + 2 B dx dy + C dy^2), d = mean2d - pixel
            ac[0] += dpower * (-(co[0] * p.dx + co[1] * p.dy));
            ac[1] += dpower * (-(co[1] * p.dx + co[2] * p.dy));
            ac[2] += dpower * (-0.5 * p.dx * p.dx);
            ac[3] += dpower * (-p.dx * p.dy);
            ac[4] += dpower * (-0.5 * p.dy * p.dy);
          }
        }
        if (sens && std::min(mg, mgc) < cutoff) {
          // flag every entry this pixel visited (ne of them) whose alpha is at or near the filter threshold
          for (uint32_t k = 0; k < (uint32_t)ne; k++) {
            const uint32_t id = sorted_ids[s + k];
            const double dx = means2d[2 * (int64_t)id] - px, dy = means2d[2 * (int64_t)id + 1] - py;
            const double* co = conic_opacity + 4 * (int64_t)id;
            const double power = -0.5 * (co[0] * dx * dx + 2.0 * co[1] * dx * dy + co[2] * dy * dy);
            const double alpha = std::min(ALPHA_MAX, co[3] * std::exp(std::min(power, 0.0)));
            if (alpha >= (1.0 - cutoff) * ALPHA_MIN) sn[k]++;
          }
        }
      }
    for (uint32_t k = 0; k < n; k++) {
      const int64_t id = sorted_ids[s + k];
      const double* ac = acc.data() + (size_t)k * 10;
      bool any = false;
      for (int j = 0; j < 10; j++) any |= ac[j] != 0.0;
      if (any) {
#pragma omp atomic
        dL_dmeans2d[2 * id] += ac[0];
#pragma omp atomic
        dL_dmeans2d[2 * id + 1] += ac[1];
#pragma omp atomic
        dL_dconic[3 * id] += ac[2];
#pragma omp atomic
        dL_dconic[3 * id + 1] += ac[3];
#pragma omp atomic
        dL_dconic[3 * id + 2] += ac[4];
#pragma omp atomic
        dL_dopacity[id] += ac[5];
#pragma omp atomic
        dL_drgb[3 * id] += ac[6];
#pragma omp atomic
        dL_drgb[3 * id + 1] += ac[7];
#pragma omp atomic
        dL_drgb[3 * id + 2] += ac[8];
#pragma omp atomic
        dL_dmask[id] += ac[9];
      }
      if (sens && sn[k]) {
#pragma omp atomic
        sens[id] += sn[k];
      }
    }
  }
  if (counts) { counts[0] = tot0; counts[1] = tot1; counts[2] = tot2; counts[3] = tot3; }
  return 0;
}

// O12.  Vector-Jacobian product of O1-O8: the projection is re-run on dual numbers carrying the
// 11 derivatives w.r.t. (mean 3, log-scale 3, raw quaternion 4, opacity logit 1); the SH
// coefficients enter linearly (dL/dsh[j][k] = Y_j(dir) dL/drgb_k unless channel k clamped).
// No gradient flows through depth, radius or rect.  Culled Gaussians get zeros.
int orc_preprocess_bwd(const Cam* cam, int64_t N, const double* means, const double* log_scales, const double* quats,
                       const double* opacity_logits, const double* sh, const double* dL_dmeans2d,
                       const double* dL_dconic, const double* dL_dopacity, const double* dL_drgb, double* dL_dmeans,
                       double* dL_dlog_scales, double* dL_dquats, double* dL_dopacity_logits, double* dL_dsh) {
  const int K = (cam->sh_degree + 1) * (cam->sh_degree + 1);
  typedef Dual<11> D;
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < N; i++) {
    D p[3], ls[3], q[4], logit;
    double shd[48], Y[16];
    for (int j = 0; j < 3; j++) { p[j] = D(means[3 * i + j]); p[j].d[j] = 1; ls[j] = D(log_scales[3 * i + j]); ls[j].d[3 + j] = 1; }
    for (int j = 0; j < 4; j++) { q[j] = D(quats[4 * i + j]); q[j].d[6 + j] = 1; }
    logit = D(opacity_logits[i]);
    logit.d[10] = 1;
    for (int j = 0; j < 3 * K; j++) shd[j] = sh[(int64_t)3 * K * i + j];
    Splat<D> s;
    project<D>(*cam, p, ls, q, logit, shd, s, Y);
    double grad[11];
    for (int j = 0; j < 11; j++) grad[j] = 0;
    double* gsh = dL_dsh + (int64_t)3 * K * i;
    for (int j = 0; j < 3 * K; j++) gsh[j] = 0;
    if (!s.culled) {
      const D* outs[9] = {&s.m2x, &s.m2y, &s.A, &s.B, &s.C, &s.o, &s.rgb[0], &s.rgb[1], &s.rgb[2]};
      const double up[9] = {dL_dmeans2d[2 * i], dL_dmeans2d[2 * i + 1], dL_dconic[3 * i], dL_dconic[3 * i + 1], dL_dconic[3 * i + 2],
                            dL_dopacity[i], dL_drgb[3 * i], dL_drgb[3 * i + 1], dL_drgb[3 * i + 2]};
      for (int o = 0; o < 9; o++)
        for (int j = 0; j < 11; j++) grad[j] += up[o] * outs[o]->d[j];
      for (int j = 0; j < K; j++)
        for (int k = 0; k < 3; k++) gsh[3 * j + k] = (s.clamped >> k & 1) ? 0.0 : Y[j] * dL_drgb[3 * i + k];
    }
    for (int j = 0; j < 3; j++) { dL_dmeans[3 * i + j] = grad[j]; dL_dlog_scales[3 * i + j] = grad[3 + j]; }
    for (int j = 0; j < 4; j++) dL_dquats[4 * i + j] = grad[6 + j];
    dL_dopacity_logits[i] = grad[10];
  }
  return 0;
}

}  // extern "C"
