// =============================================================================
//  ORACLE -- TEST INFRASTRUCTURE ONLY.
//
//  Plain, slow, fp64 CPU definition of differentiable spherical rasterisation of
//  2D Gaussian surfels into a LiDAR range image (arxiv/paper_2607_04127,
//  PAPER.md:47 section 3.1 "render the Gaussian map under the same spherical
//  projection pi_s, producing (D^, A^, N^)"; section 3.4 "optimizes the
//  Gaussian parameters Theta = {mu, q, s~, alpha}"; losses Eq. 10 PAPER.md:131 and
//  Eq. 11).  The paper names the rasteriser but does not define it;
//  every reading taken here is listed in DESIGN.md section "Readings" (R1..R19, from
//  SURVEY.md 8(c-2)).
//
//  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
//  reference legs may build, load or call this file.  It shares no code with the
//  CUDA path (paper_2607_04127_b200/csrc) and neither includes the other.
//
//  Parity pins (tests/test_oracle_*.py): closed forms (single fronto-parallel
//  surfel, two coaxial surfels, early-stop stack), invariants (A = 1 - T, seam
//  shift, rigid-frame independence, q -> -q / lambda q, scale-axis swap),
//  brute == bounded bit-for-bit, fp64 central finite differences of the scalar
//  loss for the whole backward chain, q . dL/dq = 0, Euler homogeneity.
//  Parity with the *authors'* renderer: UNPINNED (the paper prints no value for
//  this path).
//
//  Build: g++ -O2 -fopenmp -ffp-contract=off -shared -fPIC (see oracle/__init__.py)
// =============================================================================
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <limits>
#include <numeric>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

constexpr double kPi = 3.14159265358979323846;
constexpr double kAlphaMin = 1.0 / 255.0;   // reading R4: alpha >= 1/255 cut-off
constexpr double kAlphaMax = 0.99;          // reading R4: 0.99 clamp
constexpr double kRho2Max = 9.0;            // reading R4: 3 sigma
constexpr double kTmin = 1e-4;              // reading R4: stop when T(1-a) < 1e-4
constexpr double kDenMin = 1e-6;            // reading R15: grazing beams skipped
constexpr double kRectEps = 1e-9;           // angular safety margin
// Fragile-set margin on rho^2 = 9: an fp32 evaluation of u, v carries
// ~2e-5 absolute error for grazing surfels (|A| ~ r/s / cos(incidence)), i.e. <~ 2e-4 on rho^2.
constexpr double kRho2Margin = 4e-4;

struct Sensor {
  int32_t H, W;
  double elev_min, elev_max, r_min, r_max;
  double T[12];  // row-major 3x4 [R|t], p_world = R p_sensor + t
};

// Per-surfel quantities in the sensor frame.
struct Prep {
  double c[3];    // centre, sensor frame
  double tu[3], tv[3], n[3];  // columns of R_ws^T R(q^)
  double s0, s1, alpha;
  double k;       // n . c
  double sgn;     // sign(k): n^f = -sgn * n faces the sensor
  double r;       // ||c|| (fp64)
  float rkey;     // (float) r : the compositing / sort key (reading R5)
  double qh[4];   // unit quaternion
  double qn;      // ||q||
  int alive;      // passed the surfel-level culls
};

inline double dot3(const double* a, const double* b) { return a[0] * b[0] + a[1] * b[1] + a[2] * b[2]; }

// ---- step 1 + 3: frames and surfel-level culls. --------------------------------
// The arithmetic order written here IS the tile-list rule of DESIGN.md (every
// operation individually rounded, fma exactly where std::fma is written): the
// CUDA path re-implements the same order independently so that keys and rects
// are bit-identical.
void prep_surfel(const double* mean, const double* quat, const double* scale, double opacity,
                 const Sensor& S, Prep& p) {
  const double* T = S.T;
  const double R00 = T[0], R01 = T[1], R02 = T[2], tx = T[3];
  const double R10 = T[4], R11 = T[5], R12 = T[6], ty = T[7];
  const double R20 = T[8], R21 = T[9], R22 = T[10], tz = T[11];
  const double dx = mean[0] - tx, dy = mean[1] - ty, dz = mean[2] - tz;
  // c = R_ws^T (mu - t_ws)
  p.c[0] = std::fma(R00, dx, std::fma(R10, dy, R20 * dz));
  p.c[1] = std::fma(R01, dx, std::fma(R11, dy, R21 * dz));
  p.c[2] = std::fma(R02, dx, std::fma(R12, dy, R22 * dz));
  const double r2 = std::fma(p.c[2], p.c[2], std::fma(p.c[1], p.c[1], p.c[0] * p.c[0]));
  p.r = std::sqrt(r2);
  p.rkey = (float)p.r;
  p.s0 = scale[0];
  p.s1 = scale[1];
  p.alpha = opacity;
  p.alive = 1;
  if (p.alpha < kAlphaMin) p.alive = 0;                                  // cull: alpha < 1/255
  if (p.rkey < (float)S.r_min || p.rkey > (float)S.r_max) p.alive = 0;    // cull: range gate on the key (R16)
  const double smax = std::max(p.s0, p.s1);
  if (p.r <= 3.0 * smax) p.alive = 0;                                    // cull: sensor inside the 3 sigma ball (R15)
  if (!(p.s0 > 0.0) || !(p.s1 > 0.0)) p.alive = 0;                        // degenerate scale
  // unit quaternion
  const double qw = quat[0], qx = quat[1], qy = quat[2], qz = quat[3];
  const double qn2 = std::fma(qz, qz, std::fma(qy, qy, std::fma(qx, qx, qw * qw)));
  p.qn = std::sqrt(qn2);
  if (!(p.qn > 0.0) || !std::isfinite(p.qn)) {
    p.alive = 0;
    p.qn = 1.0;
  }
  const double w = qw / p.qn, x = qx / p.qn, y = qy / p.qn, z = qz / p.qn;
  p.qh[0] = w; p.qh[1] = x; p.qh[2] = y; p.qh[3] = z;
  const double xx = x * x, yy = y * y, zz = z * z;
  const double xy = x * y, xz = x * z, yz = y * z, wx = w * x, wy = w * y, wz = w * z;
  // columns e0, e1, e2 of R(q^)  (step 1; e0 = in-plane major axis)
  const double e0[3] = {1.0 - 2.0 * (yy + zz), 2.0 * (xy + wz), 2.0 * (xz - wy)};
  const double e1[3] = {2.0 * (xy - wz), 1.0 - 2.0 * (xx + zz), 2.0 * (yz + wx)};
  const double e2[3] = {2.0 * (xz + wy), 2.0 * (yz - wx), 1.0 - 2.0 * (xx + yy)};
  const double* e[3] = {e0, e1, e2};
  double* out[3] = {p.tu, p.tv, p.n};
  for (int j = 0; j < 3; ++j) {
    out[j][0] = std::fma(R00, e[j][0], std::fma(R10, e[j][1], R20 * e[j][2]));
    out[j][1] = std::fma(R01, e[j][0], std::fma(R11, e[j][1], R21 * e[j][2]));
    out[j][2] = std::fma(R02, e[j][0], std::fma(R12, e[j][1], R22 * e[j][2]));
  }
  p.k = dot3(p.n, p.c);
  p.sgn = (p.k > 0.0) ? 1.0 : ((p.k < 0.0) ? -1.0 : 0.0);
  if (!std::isfinite(p.r) || !std::isfinite(p.k)) p.alive = 0;
}

// ---- step 2: beams --------------------------------------------------------------
struct Beams {
  int H, W;
  std::vector<double> cphi, sphi, cth, sth, phi, th;
  explicit Beams(const Sensor& S) : H(S.H), W(S.W) {
    const double dphi = 2.0 * kPi / W, dth = (S.elev_max - S.elev_min) / H;
    cphi.resize(W); sphi.resize(W); phi.resize(W);
    cth.resize(H); sth.resize(H); th.resize(H);
    for (int i = 0; i < W; ++i) { phi[i] = -kPi + (i + 0.5) * dphi; cphi[i] = std::cos(phi[i]); sphi[i] = std::sin(phi[i]); }
    for (int j = 0; j < H; ++j) { th[j] = S.elev_max - (j + 0.5) * dth; cth[j] = std::cos(th[j]); sth[j] = std::sin(th[j]); }
  }
  void dir(int j, int i, double* d) const { d[0] = cth[j] * cphi[i]; d[1] = cth[j] * sphi[i]; d[2] = sth[j]; }
};

// ---- step 4: order ---------------------------------------------------------------
std::vector<int> sorted_alive(const std::vector<Prep>& P) {
  std::vector<int> order;
  order.reserve(P.size());
  for (size_t i = 0; i < P.size(); ++i) if (P[i].alive) order.push_back((int)i);
  std::stable_sort(order.begin(), order.end(), [&](int a, int b) { return P[a].rkey < P[b].rkey; });
  return order;  // ties keep ascending surfel index (stable, input ascending)
}

// One applied (pixel, surfel) pair.
struct Contrib {
  int id;
  double a, G, tau, u, v, den, T, w;
  double h[3];
  bool clamped;
};

struct PixelOut {
  double D = 0, A = 0, N[3] = {0, 0, 0};
  int ncontrib = 0;
  int fragile = 0;
  int stopped = 0;      // early stop fired
  long in3sigma = 0;    // pairs with rho2 <= 9 met before the stop
  long evaluated = 0;   // candidates visited before the stop
};

// ---- step 5: one pixel, front to back over `cand` (surfel ids in key order) ------
void composite_pixel(const double* d, const int* cand, long ncand, const Prep* P, PixelOut& o,
                     std::vector<Contrib>* rec) {
  double T = 1.0;
  for (long q = 0; q < ncand; ++q) {
    const Prep& p = P[cand[q]];
    o.evaluated++;
    const double den = dot3(p.n, d);
    // a grazing-beam decision is fragile only if the pair could otherwise contribute
    const bool den_frag = std::fabs(std::fabs(den) - kDenMin) < 0.1 * kDenMin;
    if (std::fabs(den) < kDenMin && !(den_frag && den != 0.0)) continue;
    const double tau = p.k / den;
    if (tau <= 0.0) continue;
    const double h[3] = {tau * d[0] - p.c[0], tau * d[1] - p.c[1], tau * d[2] - p.c[2]};
    const double u = dot3(p.tu, h) / p.s0;
    const double v = dot3(p.tv, h) / p.s1;
    const double rho2 = u * u + v * v;
    if (den_frag && rho2 <= kRho2Max + kRho2Margin) o.fragile = 1;
    if (std::fabs(den) < kDenMin) continue;
    if (std::fabs(rho2 - kRho2Max) < kRho2Margin) o.fragile = 1;
    if (rho2 > kRho2Max) continue;
    o.in3sigma++;
    const double G = std::exp(-0.5 * rho2);
    const double araw = p.alpha * G;
    const bool clamped = araw > kAlphaMax;
    const double a = clamped ? kAlphaMax : araw;
    if (std::fabs(araw - kAlphaMax) < 1e-6) o.fragile = 1;
    if (std::fabs(a - kAlphaMin) < 1e-6) o.fragile = 1;
    if (a < kAlphaMin) continue;
    const double test = T * (1.0 - a);
    if (std::fabs(test - kTmin) < 1e-7) o.fragile = 1;
    if (test < kTmin) { o.stopped = 1; break; }   // stop; this surfel is NOT applied
    const double w = T * a;
    o.D += w * tau;
    o.A += w;
    o.N[0] += w * (-p.sgn * p.n[0]);
    o.N[1] += w * (-p.sgn * p.n[1]);
    o.N[2] += w * (-p.sgn * p.n[2]);
    o.ncontrib++;
    if (rec) {
      Contrib cb;
      cb.id = cand[q]; cb.a = a; cb.G = G; cb.tau = tau; cb.u = u; cb.v = v; cb.den = den; cb.T = T; cb.w = w;
      cb.h[0] = h[0]; cb.h[1] = h[1]; cb.h[2] = h[2]; cb.clamped = clamped;
      rec->push_back(cb);
    }
    T = test;
  }
}

// ---- step 9: `bounded` mode candidate lists ---------------------------------------
// A surfel is dropped from a pixel's candidate list only when an fp64 bounding-cap
// test proves rho2 > 9: every point of the 3 sigma ellipse lies within smax3 = 3 max(s)
// of c, so its direction is within gamma = asin(smax3 / r) of c^.
struct CandLists {
  std::vector<long> start;  // per pixel, H*W + 1
  std::vector<int> ids;
};

CandLists build_candidates(const Sensor& S, const Beams& B, const std::vector<Prep>& P, const std::vector<int>& order) {
  const int H = S.H, W = S.W;
  const double dphi = 2.0 * kPi / W, dth = (S.elev_max - S.elev_min) / H;
  // pass 1: count
  std::vector<long> count((size_t)H * W + 1, 0);
  struct Win { int j0, j1, i0, ni; double cg; double ch[3]; };
  std::vector<Win> wins(order.size());
  for (size_t q = 0; q < order.size(); ++q) {
    const Prep& p = P[order[q]];
    Win& w = wins[q];
    const double sm3 = 3.0 * std::max(p.s0, p.s1);
    double sg = sm3 / p.r;
    if (sg > 1.0) sg = 1.0;
    const double gamma = std::asin(sg) + 1e-9;
    w.cg = std::cos(gamma);
    w.ch[0] = p.c[0] / p.r; w.ch[1] = p.c[1] / p.r; w.ch[2] = p.c[2] / p.r;
    const double thc = std::asin(std::max(-1.0, std::min(1.0, w.ch[2])));
    // rows with |theta_j - thc| <= gamma (+ one row of slack)
    int j0 = (int)std::floor((S.elev_max - (thc + gamma)) / dth - 0.5) - 1;
    int j1 = (int)std::ceil((S.elev_max - (thc - gamma)) / dth - 0.5) + 1;
    w.j0 = std::max(0, j0); w.j1 = std::min(H - 1, j1);
    // columns: all, unless the cap stays clear of the poles
    if (std::fabs(thc) + gamma >= 0.5 * kPi - 1e-6) { w.i0 = 0; w.ni = W; }
    else {
      const double hw = std::asin(std::min(1.0, std::sin(gamma) / std::cos(thc))) + 1e-9;
      const double phc = std::atan2(w.ch[1], w.ch[0]);
      long a = (long)std::floor((phc - hw + kPi) / dphi - 0.5) - 1;
      long b = (long)std::ceil((phc + hw + kPi) / dphi - 0.5) + 1;
      long ni = b - a + 1;
      if (ni >= W) { w.i0 = 0; w.ni = W; }
      else { w.i0 = (int)(((a % W) + W) % W); w.ni = (int)ni; }
    }
  }
  auto for_each_pixel = [&](size_t q, auto&& fn) {
    const Win& w = wins[q];
    for (int j = w.j0; j <= w.j1; ++j)
      for (int t = 0; t < w.ni; ++t) {
        int i = w.i0 + t; if (i >= W) i -= W;
        double d[3]; B.dir(j, i, d);
        if (dot3(d, w.ch) >= w.cg) fn((size_t)j * W + i);
      }
  };
  for (size_t q = 0; q < order.size(); ++q) for_each_pixel(q, [&](size_t px) { count[px + 1]++; });
  CandLists L;
  L.start.assign((size_t)H * W + 1, 0);
  for (size_t px = 0; px < (size_t)H * W; ++px) L.start[px + 1] = L.start[px] + count[px + 1];
  L.ids.resize((size_t)L.start.back());
  std::vector<long> fill(L.start.begin(), L.start.end() - 1);
  for (size_t q = 0; q < order.size(); ++q) for_each_pixel(q, [&](size_t px) { L.ids[(size_t)fill[px]++] = order[q]; });
  return L;
}

struct Scene {
  Sensor S;
  std::vector<Prep> P;
  std::vector<int> order;
  Scene(int64_t N, const double* mean, const double* quat, const double* scale, const double* opacity, const Sensor* s)
      : S(*s), P((size_t)N) {
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < N; ++i) prep_surfel(mean + 3 * i, quat + 4 * i, scale + 2 * i, opacity[i], S, P[(size_t)i]);
    order = sorted_alive(P);
  }
};

}  // namespace

extern "C" {

int lgs_oracle_num_threads() {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

// -----------------------------------------------------------------------------
// Forward.  mode 0 = brute (every pixel x every surviving
// surfel), 1 = bounded (same arithmetic, bounding-cap candidate lists).
// check_rects (optional, int32 [N,4] = col_min, ncols, row_min, row_max): counts
// contributing pairs that fall outside the surfel's rect into stats[5] (the
// conservativeness check of the tile-list rule).
// stats: [0] surviving surfels, [1] contributing pairs I_c, [2] pairs with rho2<=9
// met before the stop, [3] candidates visited, [4] fragile pixels, [5] rect violations,
// [6] pixels that stopped early.
// -----------------------------------------------------------------------------
int lgs_oracle_forward(int64_t N, const double* mean, const double* quat, const double* scale, const double* opacity,
                       const Sensor* sensor, int mode, double* out_range, double* out_alpha, double* out_normal,
                       int32_t* out_ncontrib, uint8_t* out_fragile, const int32_t* check_rects, int64_t* stats) {
  Scene sc(N, mean, quat, scale, opacity, sensor);
  const int H = sc.S.H, W = sc.S.W;
  Beams B(sc.S);
  CandLists L;
  if (mode == 1) L = build_candidates(sc.S, B, sc.P, sc.order);
  long Ic = 0, I3 = 0, Iev = 0, nfrag = 0, nviol = 0, nstop = 0;
#pragma omp parallel for schedule(dynamic, 64) reduction(+ : Ic, I3, Iev, nfrag, nviol, nstop)
  for (long px = 0; px < (long)H * W; ++px) {
    const int j = (int)(px / W), i = (int)(px % W);
    double d[3];
    B.dir(j, i, d);
    PixelOut o;
    std::vector<Contrib> rec;
    const int* cand = mode == 1 ? L.ids.data() + L.start[px] : sc.order.data();
    const long nc = mode == 1 ? L.start[px + 1] - L.start[px] : (long)sc.order.size();
    composite_pixel(d, cand, nc, sc.P.data(), o, check_rects ? &rec : nullptr);
    out_range[px] = o.D;
    out_alpha[px] = o.A;
    if (out_normal) {
      out_normal[px] = o.N[0];
      out_normal[(size_t)H * W + px] = o.N[1];
      out_normal[2 * (size_t)H * W + px] = o.N[2];
    }
    if (out_ncontrib) out_ncontrib[px] = o.ncontrib;
    if (out_fragile) out_fragile[px] = (uint8_t)o.fragile;
    Ic += o.ncontrib; I3 += o.in3sigma; Iev += o.evaluated; nfrag += o.fragile; nstop += o.stopped;
    if (check_rects)
      for (const Contrib& cb : rec) {
        const int32_t* r = check_rects + 4 * (size_t)cb.id;
        int dc = i - r[0]; if (dc < 0) dc += W;
        if (!(r[1] > 0 && dc < r[1] && j >= r[2] && j <= r[3])) nviol++;
      }
  }
  if (stats) {
    stats[0] = (int64_t)sc.order.size(); stats[1] = Ic; stats[2] = I3; stats[3] = Iev;
    stats[4] = nfrag; stats[5] = nviol; stats[6] = nstop;
  }
  return 0;
}

// -----------------------------------------------------------------------------
// Footprint census for the roofline's work counts ("N_fp = surfels with a non-empty footprint").
// touched[i] = 1 iff some beam of the grid meets the plane of surviving surfel i inside its 3 sigma ellipse under the
// cut-offs of step 5 that concern the pair alone (|den| >= den_min, tau > 0, rho2 <= 9); what other surfels do to the
// beam (occlusion, the early stop) and the opacity threshold on alpha G play no part.  Same expressions as
// composite_pixel, over the bounded candidate lists (which drop a pair only when rho2 > 9 is proven).  A count, not a
// rendered value: nothing of the forward / backward depends on it.  Returns N_fp.
// -----------------------------------------------------------------------------
int64_t lgs_oracle_footprint(int64_t N, const double* mean, const double* quat, const double* scale,
                             const double* opacity, const Sensor* sensor, uint8_t* touched) {
  Scene sc(N, mean, quat, scale, opacity, sensor);
  const int H = sc.S.H, W = sc.S.W;
  Beams B(sc.S);
  const CandLists L = build_candidates(sc.S, B, sc.P, sc.order);
  std::vector<uint8_t> mark((size_t)N, 0);
#pragma omp parallel for schedule(dynamic, 64)
  for (long px = 0; px < (long)H * W; ++px) {
    const int j = (int)(px / W), i = (int)(px % W);
    double d[3];
    B.dir(j, i, d);
    for (long q = L.start[px]; q < L.start[px + 1]; ++q) {
      const int id = L.ids[q];
      const Prep& p = sc.P[id];
      const double den = dot3(p.n, d);
      if (std::fabs(den) < kDenMin) continue;
      const double tau = p.k / den;
      if (tau <= 0.0) continue;
      const double h[3] = {tau * d[0] - p.c[0], tau * d[1] - p.c[1], tau * d[2] - p.c[2]};
      const double u = dot3(p.tu, h) / p.s0;
      const double v = dot3(p.tv, h) / p.s1;
      if (u * u + v * v > kRho2Max) continue;
#pragma omp atomic write
      mark[id] = 1;
    }
  }
  int64_t n = 0;
  for (int64_t k = 0; k < N; ++k) { n += mark[k]; if (touched) touched[k] = mark[k]; }
  return n;
}

// -----------------------------------------------------------------------------
// Backward: plain adjoint of step 5 for given upstream
// images gD = dL/dD^, gA = dL/dA^, gN = dL/dN^ ([3,H,W]); cut-offs and the stop index
// are piecewise constant.  Outputs dL/dmean [N,3], dL/dquat [N,4] (through the
// normalisation), dL/dscale [N,2], dL/dopacity [N]; culled surfels get zeros.
// -----------------------------------------------------------------------------
int lgs_oracle_backward(int64_t N, const double* mean, const double* quat, const double* scale, const double* opacity,
                        const Sensor* sensor, int mode, const double* gD, const double* gA, const double* gN,
                        double* g_mean, double* g_quat, double* g_scale, double* g_opacity, double* cond) {
  // cond (optional, [N,4], diagnostic only): per surfel and parameter group (mean, quat, scale,
  // opacity) the sum over pairs of |contribution| x kappa.  kappa bounds, to first order, how much
  // a relative perturbation eps of every evaluated alpha a_l of the pixel moves abar_i relative
  // to |abar_i|:  abar_i = T_i x_i - T_i sum_{j>i} omega_j x_j with T_i = prod_{l<i}(1 - a_l),
  // omega_j = a_j prod_{i<l<j}(1 - a_l), and d(1 - a_l)/(1 - a_l) = -eps a_l/(1 - a_l), hence
  //   |d abar_i| <= eps (1 + sum_l 1/((1 - a_l) |d.n_l|)) (|T_i x_i| + sum_{j>i} w_j |x_j| / (1 - a_i)),
  // kappa = that bracket / |abar_i| >= 1 (error <~ k eps cond).  Two things make the chain
  // ill-conditioned: near-opaque contributors (1/(1 - a) reaches 100) and grazing incidence, where
  // u = (d.A_u)/(d.n) divides two nearly cancelling sums, so that the relative error of an evaluated
  // alpha grows like 1/|d.n| (with the cut-off at |d.n| = 1e-6 this is unbounded in principle).
  // cond never feeds back into the gradients.
  Scene sc(N, mean, quat, scale, opacity, sensor);
  const int H = sc.S.H, W = sc.S.W;
  const size_t HW = (size_t)H * W;
  Beams B(sc.S);
  CandLists L;
  if (mode == 1) L = build_candidates(sc.S, B, sc.P, sc.order);
  // per-surfel adjoints: cbar(3) nbar(3) tubar(3) tvbar(3) s0bar s1bar alphabar
  std::vector<double> acc((size_t)N * 15, 0.0);
  if (cond) std::fill(cond, cond + 4 * (size_t)N, 0.0);
#pragma omp parallel for schedule(dynamic, 64)
  for (long px = 0; px < (long)HW; ++px) {
    const int j = (int)(px / W), i = (int)(px % W);
    const double gd = gD ? gD[px] : 0.0, ga = gA ? gA[px] : 0.0;
    const double gn[3] = {gN ? gN[px] : 0.0, gN ? gN[HW + px] : 0.0, gN ? gN[2 * HW + px] : 0.0};
    if (gd == 0.0 && ga == 0.0 && gn[0] == 0.0 && gn[1] == 0.0 && gn[2] == 0.0) continue;
    double d[3];
    B.dir(j, i, d);
    PixelOut o;
    std::vector<Contrib> rec;
    const int* cand = mode == 1 ? L.ids.data() + L.start[px] : sc.order.data();
    const long nc = mode == 1 ? L.start[px + 1] - L.start[px] : (long)sc.order.size();
    composite_pixel(d, cand, nc, sc.P.data(), o, &rec);
    const int m = (int)rec.size();
    // step 7: x_i, suffix sums S_i = sum_{j>i} w_j x_j
    std::vector<double> x(m), Ssuf(m);
    for (int q = 0; q < m; ++q) {
      const Prep& p = sc.P[rec[q].id];
      const double nf[3] = {-p.sgn * p.n[0], -p.sgn * p.n[1], -p.sgn * p.n[2]};
      x[q] = gd * rec[q].tau + ga + dot3(gn, nf);
    }
    double run = 0.0;
    for (int q = m - 1; q >= 0; --q) { Ssuf[q] = run; run += rec[q].w * x[q]; }
    std::vector<double> Sabs;      // cond only: sum_{j>q} w_j |x_j|
    double amp = 1.0;              // cond only: 1 + sum_l 1 / ((1 - a_l) min(1, |d.n_l|))
    if (cond) {
      Sabs.resize(m);
      double ra = 0.0;
      for (int q = m - 1; q >= 0; --q) { Sabs[q] = ra; ra += rec[q].w * std::fabs(x[q]); amp += 1.0 / ((1.0 - rec[q].a) * std::min(1.0, std::fabs(rec[q].den))); }
    }
    for (int q = 0; q < m; ++q) {
      const Contrib& cb = rec[q];
      const Prep& p = sc.P[cb.id];
      double abar = cb.T * x[q] - Ssuf[q] / (1.0 - cb.a);
      const double taubar = cb.w * gd;
      const double nfbar[3] = {cb.w * gn[0], cb.w * gn[1], cb.w * gn[2]};
      if (cb.clamped) abar = 0.0;              // true derivative of min(0.99, .) (reading R17)
      const double alphabar = cb.G * abar;
      const double Gbar = p.alpha * abar;
      const double ubar = -cb.u * cb.G * Gbar;
      const double vbar = -cb.v * cb.G * Gbar;
      // step 8: plain adjoint to the sensor-frame surfel quantities
      double hbar[3], cbar[3], nbar[3], tubar[3], tvbar[3];
      for (int a = 0; a < 3; ++a) hbar[a] = ubar * p.tu[a] / p.s0 + vbar * p.tv[a] / p.s1;
      const double tautot = taubar + dot3(hbar, d);
      for (int a = 0; a < 3; ++a) {
        cbar[a] = -hbar[a] + tautot * p.n[a] / cb.den;
        nbar[a] = -tautot * cb.h[a] / cb.den - p.sgn * nfbar[a];
        tubar[a] = ubar * cb.h[a] / p.s0;
        tvbar[a] = vbar * cb.h[a] / p.s1;
      }
      const double s0bar = -ubar * cb.u / p.s0;
      const double s1bar = -vbar * cb.v / p.s1;
      double* A = acc.data() + (size_t)cb.id * 15;
      const double vals[15] = {cbar[0], cbar[1], cbar[2], nbar[0], nbar[1], nbar[2], tubar[0], tubar[1], tubar[2],
                               tvbar[0], tvbar[1], tvbar[2], s0bar, s1bar, alphabar};
      for (int a = 0; a < 15; ++a) {
#pragma omp atomic
        A[a] += vals[a];
      }
      if (cond) {
        const double t1 = std::fabs(cb.T * x[q]), t2 = Sabs[q] / (1.0 - cb.a);
        const double kap = (abar != 0.0) ? amp * (t1 + t2) / std::fabs(abar) : 1.0;
        // the geometric terms scale with abar (times kappa); the direct terms (taubar, nfbar) do not
        const double geo = std::sqrt(dot3(hbar, hbar)) * kap + std::fabs(tautot / cb.den);
        const double rot = (std::sqrt(dot3(tubar, tubar)) + std::sqrt(dot3(tvbar, tvbar))) * kap +
                           std::fabs(tautot / cb.den) * std::sqrt(dot3(cb.h, cb.h)) + std::sqrt(dot3(nfbar, nfbar));
        const double cv[4] = {geo, 2.0 * rot / p.qn, (std::fabs(s0bar) + std::fabs(s1bar)) * kap, std::fabs(alphabar) * kap};
        for (int a = 0; a < 4; ++a) {
#pragma omp atomic
          cond[4 * (size_t)cb.id + a] += cv[a];
        }
      }
    }
  }
  // step 8 (cont.): sensor frame -> world parameters
  const double* T = sc.S.T;
  const double R[3][3] = {{T[0], T[1], T[2]}, {T[4], T[5], T[6]}, {T[8], T[9], T[10]}};
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < N; ++i) {
    const Prep& p = sc.P[(size_t)i];
    double* gm = g_mean + 3 * i; double* gq = g_quat + 4 * i; double* gs = g_scale + 2 * i;
    gm[0] = gm[1] = gm[2] = 0; gq[0] = gq[1] = gq[2] = gq[3] = 0; gs[0] = gs[1] = 0; g_opacity[i] = 0;
    if (!p.alive) continue;
    const double* A = acc.data() + (size_t)i * 15;
    // mu_bar = R_ws c_bar
    for (int a = 0; a < 3; ++a) gm[a] = R[a][0] * A[0] + R[a][1] * A[1] + R[a][2] * A[2];
    // M = R_ws [tu_bar tv_bar n_bar] = dL/dR(q^), M[row][col]
    double M[3][3];
    for (int a = 0; a < 3; ++a) {
      M[a][0] = R[a][0] * A[6] + R[a][1] * A[7] + R[a][2] * A[8];
      M[a][1] = R[a][0] * A[9] + R[a][1] * A[10] + R[a][2] * A[11];
      M[a][2] = R[a][0] * A[3] + R[a][1] * A[4] + R[a][2] * A[5];
    }
    const double w = p.qh[0], x = p.qh[1], y = p.qh[2], z = p.qh[3];
    // 1-indexed M_ij of SURVEY step 8 -> M[i-1][j-1]
    double gh[4];
    gh[0] = 2.0 * (x * (M[2][1] - M[1][2]) + y * (M[0][2] - M[2][0]) + z * (M[1][0] - M[0][1]));
    gh[1] = 2.0 * (y * (M[0][1] + M[1][0]) + z * (M[0][2] + M[2][0]) - 2.0 * x * (M[1][1] + M[2][2]) + w * (M[2][1] - M[1][2]));
    gh[2] = 2.0 * (x * (M[0][1] + M[1][0]) + z * (M[1][2] + M[2][1]) - 2.0 * y * (M[0][0] + M[2][2]) + w * (M[0][2] - M[2][0]));
    gh[3] = 2.0 * (x * (M[0][2] + M[2][0]) + y * (M[1][2] + M[2][1]) - 2.0 * z * (M[0][0] + M[1][1]) + w * (M[1][0] - M[0][1]));
    // through q^ = q / ||q||
    const double qg = p.qh[0] * gh[0] + p.qh[1] * gh[1] + p.qh[2] * gh[2] + p.qh[3] * gh[3];
    for (int a = 0; a < 4; ++a) gq[a] = (gh[a] - p.qh[a] * qg) / p.qn;
    gs[0] = A[12]; gs[1] = A[13];
    g_opacity[i] = A[14];
  }
  return 0;
}

// -----------------------------------------------------------------------------
// Loss stage: masked L1 range (Eq. 10 left),
// cosine loss vs N_g-icp over Omega_N, cosine loss vs N_surf from
// the rendered range over Omega_S, normalised by |Omega_M| (Eq. 11).
// L = L_depth + lambda_n (lambda_ng L_ng + lambda_ns L_ns).
// out_losses: [0] L, [1] L_depth, [2] L_ng, [3] L_ns.  out_counts: |Omega_M|, |Omega_N|, |Omega_S|.
// sign_fragile: pixels whose L1 sign is decided by |D^ - D| < 1e-5 max(D, 1).
// -----------------------------------------------------------------------------
int lgs_oracle_loss(const Sensor* sensor, const double* range, const double* alpha, const double* normal,
                    const double* target_range, const double* target_normal, const uint8_t* keep_mask,
                    double lambda_n, double lambda_ng, double lambda_ns, int detach_surf,
                    double* out_losses, int64_t* out_counts, double* gD, double* gA, double* gN,
                    uint8_t* sign_fragile) {
  (void)alpha;
  const Sensor& S = *sensor;
  const int H = S.H, W = S.W;
  const size_t HW = (size_t)H * W;
  Beams B(S);
  std::vector<uint8_t> inM(HW), inN(HW, 0);
  long nM = 0, nN = 0, nS = 0;
  for (size_t px = 0; px < HW; ++px) {
    inM[px] = (target_range[px] > 0.0) && (!keep_mask || keep_mask[px] != 0);
    nM += inM[px];
    if (inM[px] && target_normal) {
      const double n2 = target_normal[px] * target_normal[px] + target_normal[HW + px] * target_normal[HW + px] +
                        target_normal[2 * HW + px] * target_normal[2 * HW + px];
      inN[px] = n2 > 0.0;
      nN += inN[px];
    }
  }
  for (size_t px = 0; px < HW; ++px) { gD[px] = 0; gA[px] = 0; gN[px] = gN[HW + px] = gN[2 * HW + px] = 0; if (sign_fragile) sign_fragile[px] = 0; }
  double Ld = 0, Lng = 0, Lns = 0;
  if (nM > 0) {
    for (size_t px = 0; px < HW; ++px) {
      if (!inM[px]) continue;
      const double e = range[px] - target_range[px];
      Ld += std::fabs(e);
      gD[px] += ((e > 0) - (e < 0)) / (double)nM;
      if (sign_fragile && std::fabs(e) < 1e-5 * std::max(target_range[px], 1.0)) sign_fragile[px] = 1;
    }
    Ld /= (double)nM;
    if (nN > 0) {
      for (size_t px = 0; px < HW; ++px) {
        if (!inN[px]) continue;
        const double ng[3] = {target_normal[px], target_normal[HW + px], target_normal[2 * HW + px]};
        const double nh[3] = {normal[px], normal[HW + px], normal[2 * HW + px]};
        Lng += 1.0 - dot3(nh, ng);
        for (int a = 0; a < 3; ++a) gN[a * HW + px] -= lambda_n * lambda_ng * ng[a] / (double)nN;
      }
      Lng /= (double)nN;
    }
    // N_surf term
    auto X = [&](int j, int i, double* x) { double d[3]; B.dir(j, i, d); const double r = range[(size_t)j * W + i]; x[0] = r * d[0]; x[1] = r * d[1]; x[2] = r * d[2]; };
    for (int j = 1; j + 1 < H; ++j)
      for (int i = 0; i < W; ++i) {
        const int ip = (i + 1) % W, im = (i + W - 1) % W;
        const size_t px = (size_t)j * W + i;
        const size_t pe = (size_t)j * W + ip, pw = (size_t)j * W + im, pu = (size_t)(j - 1) * W + i, pd = (size_t)(j + 1) * W + i;
        if (!(inM[px] && inM[pe] && inM[pw] && inM[pu] && inM[pd])) continue;
        double xe[3], xw[3], xu[3], xd[3];
        X(j, ip, xe); X(j, im, xw); X(j - 1, i, xu); X(j + 1, i, xd);
        const double dp[3] = {xe[0] - xw[0], xe[1] - xw[1], xe[2] - xw[2]};   // d_phi X
        const double dt[3] = {xu[0] - xd[0], xu[1] - xd[1], xu[2] - xd[2]};   // d_theta X
        const double m[3] = {dp[1] * dt[2] - dp[2] * dt[1], dp[2] * dt[0] - dp[0] * dt[2], dp[0] * dt[1] - dp[1] * dt[0]};
        const double mn = std::sqrt(dot3(m, m));
        if (mn < 1e-12) continue;
        nS++;
        const double ns[3] = {-m[0] / mn, -m[1] / mn, -m[2] / mn};
        const double nh[3] = {normal[px], normal[HW + px], normal[2 * HW + px]};
        Lns += 1.0 - dot3(nh, ns);
        const double cf = lambda_n * lambda_ns / (double)nM;
        for (int a = 0; a < 3; ++a) gN[a * HW + px] -= cf * ns[a];
        if (!detach_surf) {
          // l = 1 - N^.N^s, N^s = -m/|m|  =>  dl/dm = (I - m^ m^T) N^ / |m|
          const double mh[3] = {m[0] / mn, m[1] / mn, m[2] / mn};
          const double pr = dot3(mh, nh);
          const double gm[3] = {cf * (nh[0] - pr * mh[0]) / mn, cf * (nh[1] - pr * mh[1]) / mn, cf * (nh[2] - pr * mh[2]) / mn};
          // dm = d(dp) x dt + dp x d(dt)  =>  dL/d(dp) = dt x gm ; dL/d(dt) = gm x dp
          const double Gp[3] = {dt[1] * gm[2] - dt[2] * gm[1], dt[2] * gm[0] - dt[0] * gm[2], dt[0] * gm[1] - dt[1] * gm[0]};
          const double Gt[3] = {gm[1] * dp[2] - gm[2] * dp[1], gm[2] * dp[0] - gm[0] * dp[2], gm[0] * dp[1] - gm[1] * dp[0]};
          double de[3], dw[3], du[3], dd[3];
          B.dir(j, ip, de); B.dir(j, im, dw); B.dir(j - 1, i, du); B.dir(j + 1, i, dd);
          gD[pe] += dot3(de, Gp);
          gD[pw] -= dot3(dw, Gp);
          gD[pu] += dot3(du, Gt);
          gD[pd] -= dot3(dd, Gt);
        }
      }
    Lns /= (double)nM;
  }
  out_losses[1] = Ld; out_losses[2] = Lng; out_losses[3] = Lns;
  out_losses[0] = Ld + lambda_n * (lambda_ng * Lng + lambda_ns * Lns);
  out_counts[0] = nM; out_counts[1] = nN; out_counts[2] = nS;
  return 0;
}

// -----------------------------------------------------------------------------
// List reference (rule stated in DESIGN.md "tile-list rule").
// rect (int32 [N,4]): col_min in [0,W), ncols in [0,W] (0 = culled / empty),
// row_min, row_max (inclusive).  Emission in ascending surfel index; key64 =
// (tile_id << 32) | float_bits(rkey); std::stable_sort; per-tile [start, end).
// Tiles are tile_w columns x tile_h rows (a parameter of the list structure, not of the
// arithmetic: the rect and the key do not depend on it); tile_id = tile_row * ntc + tile_col.
// Returns K (number of keys); arrays are filled only if K <= capacity.
// -----------------------------------------------------------------------------
int64_t lgs_oracle_tile_lists(int64_t N, const double* mean, const double* quat, const double* scale,
                              const double* opacity, const Sensor* sensor, int tile_w, int tile_h, int64_t capacity,
                              uint64_t* keys, uint32_t* vals, uint32_t* tile_ranges, int32_t* rects, float* rkeys) {
  const Sensor& S = *sensor;
  const int H = S.H, W = S.W;
  const int ntc = (W + tile_w - 1) / tile_w, ntr = (H + tile_h - 1) / tile_h;
  const double dphi = (2.0 * kPi) / (double)W;
  const double dth = (S.elev_max - S.elev_min) / (double)H;
  std::vector<std::pair<uint64_t, uint32_t>> kv;
  for (int64_t i = 0; i < N; ++i) {
    Prep p;
    prep_surfel(mean + 3 * i, quat + 4 * i, scale + 2 * i, opacity[i], S, p);
    int32_t* rc = rects + 4 * i;
    rc[0] = rc[1] = rc[2] = rc[3] = 0;
    if (rkeys) rkeys[i] = p.rkey;
    if (!p.alive) continue;
    // 3 sigma semi-axes in the sensor frame
    const double k0 = 3.0 * p.s0, k1 = 3.0 * p.s1;
    const double a[3] = {k0 * p.tu[0], k0 * p.tu[1], k0 * p.tu[2]};
    const double b[3] = {k1 * p.tv[0], k1 * p.tv[1], k1 * p.tv[2]};
    const double cx = p.c[0], cy = p.c[1], cz = p.c[2];
    const double rho = std::sqrt(std::fma(cy, cy, cx * cx));
    double erx = 1.0, ery = 0.0;
    if (rho > 0.0) { erx = cx / rho; ery = cy / rho; }
    const double ar = std::fma(a[1], ery, a[0] * erx), br = std::fma(b[1], ery, b[0] * erx);
    const double at = std::fma(a[1], erx, -(a[0] * ery)), bt = std::fma(b[1], erx, -(b[0] * ery));
    const double hr = std::sqrt(std::fma(br, br, ar * ar));
    const double ht = std::sqrt(std::fma(bt, bt, at * at));
    const double hz = std::sqrt(std::fma(b[2], b[2], a[2] * a[2]));
    const double rho_lo = rho - hr, rho_out = rho + hr;
    const double rho_hi = std::sqrt(std::fma(ht, ht, rho_out * rho_out));
    const double z_lo = cz - hz, z_hi = cz + hz;
    int col_min, ncols;
    double th_lo, th_hi;
    if (rho_lo > 0.0) {
      const double half = std::atan(ht / rho_lo) + kRectEps;
      const double phc = std::atan2(cy, cx);
      const double flo = std::ceil((phc - half + kPi) / dphi - 0.5);
      const double fhi = std::floor((phc + half + kPi) / dphi - 0.5);
      const double fn = fhi - flo + 1.0;
      if (!(fn >= 1.0)) continue;  // no pixel centre inside: culled
      if (fn >= (double)W) { col_min = 0; ncols = W; }
      else {
        long lo = (long)flo;
        col_min = (int)(((lo % W) + W) % W);
        ncols = (int)fn;
      }
      th_lo = std::atan2(z_lo, z_lo < 0.0 ? rho_lo : rho_hi) - kRectEps;
      th_hi = std::atan2(z_hi, z_hi > 0.0 ? rho_lo : rho_hi) + kRectEps;
    } else {
      col_min = 0; ncols = W;
      th_lo = z_lo > 0.0 ? std::atan2(z_lo, rho_hi) - kRectEps : -0.5 * kPi;
      th_hi = z_hi < 0.0 ? std::atan2(z_hi, rho_hi) + kRectEps : 0.5 * kPi;
    }
    double frlo = std::ceil((S.elev_max - th_hi) / dth - 0.5);
    double frhi = std::floor((S.elev_max - th_lo) / dth - 0.5);
    if (frlo < 0.0) frlo = 0.0;
    if (frhi > (double)(H - 1)) frhi = (double)(H - 1);
    if (!(frhi >= frlo)) continue;  // outside the vertical FOV / between rows: culled
    rc[0] = col_min; rc[1] = ncols; rc[2] = (int)frlo; rc[3] = (int)frhi;
    // tiles touched (tile columns wrap across the seam, each tile at most once)
    const int tr0 = rc[2] / tile_h, tr1 = rc[3] / tile_h;
    const int tc0 = col_min / tile_w;
    int ntcs;
    if (ncols >= W) ntcs = ntc;
    else {
      // walk the wrapped column interval and count distinct tile columns
      const int last = col_min + ncols - 1;  // may exceed W-1
      if (last < W) ntcs = last / tile_w - tc0 + 1;
      else ntcs = (ntc - tc0) + ((last - W) / tile_w + 1);
      if (ntcs > ntc) ntcs = ntc;
    }
    uint32_t kb;
    std::memcpy(&kb, &p.rkey, 4);
    for (int tr = tr0; tr <= tr1; ++tr)
      for (int t = 0; t < ntcs; ++t) {
        int tc = tc0 + t; if (tc >= ntc) tc -= ntc;
        const uint64_t tid = (uint64_t)tr * ntc + tc;
        kv.emplace_back((tid << 32) | kb, (uint32_t)i);
      }
  }
  const int64_t K = (int64_t)kv.size();
  std::stable_sort(kv.begin(), kv.end(), [](const auto& x, const auto& y) { return x.first < y.first; });
  if (K <= capacity) {
    for (int64_t q = 0; q < K; ++q) { keys[q] = kv[(size_t)q].first; vals[q] = kv[(size_t)q].second; }
  }
  if (tile_ranges) {
    const int nt = ntc * ntr;
    for (int t = 0; t < 2 * nt; ++t) tile_ranges[t] = 0;
    int64_t q = 0;
    for (int t = 0; t < nt; ++t) {
      while (q < K && (kv[(size_t)q].first >> 32) < (uint64_t)t) ++q;
      tile_ranges[2 * t] = (uint32_t)q;
      int64_t e = q;
      while (e < K && (kv[(size_t)e].first >> 32) == (uint64_t)t) ++e;
      tile_ranges[2 * t + 1] = (uint32_t)e;
      q = e;
    }
  }
  return K;
}

}  // extern "C"
