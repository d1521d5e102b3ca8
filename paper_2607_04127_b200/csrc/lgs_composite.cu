// K5 / K7 / K8: per-tile front-to-back compositing (forward), its adjoint (backward, warp
// butterfly reduction before global atomics) and the per-surfel chain rule to (mu, q, s, alpha).
//
// Steps S5, S7, S8 of SURVEY.md 8(a); north_star (3), (4).  What is rendered: PAPER.md:47 / 127
// (D^, A^, N^); cut-offs and ordering: DESIGN.md readings R3-R7, R15, R17.
//
// Pair evaluation: with the per-surfel record
//   n^f = sigma n, k^f = sigma (n.c) = -|n.c|, A_u = sigma (t_v x c)/s0, A_v = sigma (c x t_u)/s1,
// a beam d hits the surfel plane at tau = k^f/(d.n^f) with local coordinates
// u = (d.A_u)/(d.n^f), v = (d.A_v)/(d.n^f): three dot products and one reciprocal per pair.
// All arithmetic of a pair is written with explicit round-to-nearest intrinsics so that the
// forward and the backward kernel take bit-identical cut-off decisions.
#include "lgs_internal.cuh"

namespace lgs {
namespace {

constexpr int kCompThreads = 256;   // 8 warps: one 16x16 tile
constexpr int kBatch = 256;         // list entries staged per round
constexpr int kSubW = 16, kSubH = 2;  // pixels of one warp: 16 columns x 2 rows
static_assert(kSubW * kSubH == 32, "one pixel per lane");

__device__ __forceinline__ float rcp_approx(float x) {
  float y;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ float ex2_approx(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}

struct PairEval {
  float inv, u, v, G, a, tau;
  bool clamped;
};

// Tile-anchored pair evaluation.  The beam of a pixel is d_p = d_t + delta with d_t the tile's
// reference beam (kept as hi + lo floats) and delta small, exact to ~6e-9.  At staging time each
// list entry gets its values at the reference beam,
//   den0 = d_t.n^f,  pu0 = (d_t - c^).A_u,  pv0 = (d_t - c^).A_v      (c^.A_u = c^.A_v = 0 exactly),
// with c^ = c/|c| also kept as hi + lo, so the large products |A| ~ r/s only ever multiply the
// small vectors (d_t - c^) and delta.  Per pair: three 3-term fma chains and one reciprocal.
// Returns true if the pair passes every per-pair cut-off (den, 3 sigma, alpha >= 1/255).
__device__ __forceinline__ bool eval_pair(float ex, float ey, float ez, const float4& q0, const float4& q1,
                                          const float4& q2, const float4& q3, PairEval& e) {
  const float den = __fmaf_rn(ex, q0.x, __fmaf_rn(ey, q0.y, __fmaf_rn(ez, q0.z, q2.w)));
  if (!(den < -LGS_DEN_MIN)) return false;        // grazing or back-facing beam (tau <= 0)
  e.inv = rcp_approx(den);
  const float pu = __fmaf_rn(ex, q1.x, __fmaf_rn(ey, q1.y, __fmaf_rn(ez, q1.z, q3.x)));
  const float pv = __fmaf_rn(ex, q2.x, __fmaf_rn(ey, q2.y, __fmaf_rn(ez, q2.z, q3.y)));
  e.u = __fmul_rn(pu, e.inv);
  e.v = __fmul_rn(pv, e.inv);
  const float rho2 = __fmaf_rn(e.u, e.u, __fmul_rn(e.v, e.v));
  if (!(rho2 <= LGS_RHO2_MAX)) return false;
  e.G = ex2_approx(__fmul_rn(rho2, -0.72134752044448170368f));   // exp(-rho2/2)
  const float araw = __fmul_rn(q1.w, e.G);
  e.clamped = araw > LGS_ALPHA_MAX;
  e.a = e.clamped ? LGS_ALPHA_MAX : araw;
  if (!(e.a >= LGS_ALPHA_MIN)) return false;
  e.tau = __fmul_rn(q0.w, e.inv);
  return true;
}

struct TileGeom {
  int col, row, col0w, row0w, subw, subh;
  bool inside;
  float ex, ey, ez;        // delta = d_p - d_t
  float dx, dy, dz;        // d_p rounded to fp32 (used only for gradient accumulation)
  float thx, thy, thz, tlx, tly, tlz;   // d_t = hi + lo
};

__device__ __forceinline__ void beam64(const double* tab, int W, int H, int row, int col, double* d) {
  const double cph = tab[col], sph = tab[W + col], cth = tab[2 * W + row], sth = tab[2 * W + H + row];
  d[0] = cth * cph; d[1] = cth * sph; d[2] = sth;
}

__device__ __forceinline__ TileGeom tile_geom(int tile, const SensorDev& S, const double* tab, int warp, int lane) {
  TileGeom g;
  const int tr = tile / S.ntc, tc = tile - tr * S.ntc;
  constexpr int wx = kTile / kSubW;
  g.col0w = tc * kTile + (warp % wx) * kSubW;
  g.row0w = tr * kTile + (warp / wx) * kSubH;
  g.col = g.col0w + (lane % kSubW);
  g.row = g.row0w + (lane / kSubW);
  g.inside = g.col < S.W && g.row < S.H;
  g.subw = min(kSubW, S.W - g.col0w);
  g.subh = min(kSubH, S.H - g.row0w);
  double dt[3], dp[3];
  beam64(tab, S.W, S.H, min(tr * kTile + kTile / 2, S.H - 1), min(tc * kTile + kTile / 2, S.W - 1), dt);
  g.thx = (float)dt[0]; g.thy = (float)dt[1]; g.thz = (float)dt[2];
  g.tlx = (float)(dt[0] - (double)g.thx); g.tly = (float)(dt[1] - (double)g.thy); g.tlz = (float)(dt[2] - (double)g.thz);
  beam64(tab, S.W, S.H, min(g.row, S.H - 1), min(g.col, S.W - 1), dp);
  g.ex = (float)(dp[0] - dt[0]); g.ey = (float)(dp[1] - dt[1]); g.ez = (float)(dp[2] - dt[2]);
  g.dx = (float)dp[0]; g.dy = (float)dp[1]; g.dz = (float)dp[2];
  return g;
}

// Does the (wrapped) rect of a surfel overlap this warp's pixel block?
__device__ __forceinline__ bool rect_hits(unsigned int rx, unsigned int ry, const TileGeom& g, int W) {
  const int col_min = (int)(rx & 0xffffu), ncols = (int)(rx >> 16);
  const int row_min = (int)(ry & 0xffffu), row_max = (int)(ry >> 16);
  if (row_max < g.row0w || row_min >= g.row0w + g.subh) return false;
  int rel = g.col0w - col_min;
  if (rel < 0) rel += W;
  if (rel < ncols) return true;
  int rel2 = col_min - g.col0w;
  if (rel2 < 0) rel2 += W;
  return rel2 < g.subw;
}

// Staged (shared-memory) form of one list entry: 4 x float4, read by broadcast.
//   q0 = n^f.xyz, k^f | q1 = A_u.xyz, alpha | q2 = A_v.xyz, den0 | q3 = pu0, pv0, rect.x, rect.y
struct Stage {
  float4 q0[kBatch], q1[kBatch], q2[kBatch], q3[kBatch];
};

__device__ __forceinline__ void stage_entry(Stage& s, int slot, const float4* __restrict__ rec, const TileGeom& g) {
  const float4 r0 = __ldg(rec), r1 = __ldg(rec + 1), r2 = __ldg(rec + 2), r3 = __ldg(rec + 3), r4 = __ldg(rec + 4);
  // e = d_t - c^ in two-float arithmetic (the hi parts nearly cancel, the lo parts restore the bits)
  const float ex = __fadd_rn(__fsub_rn(g.thx, r3.x), __fsub_rn(g.tlx, r4.x));
  const float ey = __fadd_rn(__fsub_rn(g.thy, r3.y), __fsub_rn(g.tly, r4.y));
  const float ez = __fadd_rn(__fsub_rn(g.thz, r3.z), __fsub_rn(g.tlz, r4.z));
  const float den0 = __fmaf_rn(g.thx, r0.x, __fmaf_rn(g.thy, r0.y, __fmul_rn(g.thz, r0.z)));
  const float pu0 = __fmaf_rn(ex, r1.x, __fmaf_rn(ey, r1.y, __fmul_rn(ez, r1.z)));
  const float pv0 = __fmaf_rn(ex, r2.x, __fmaf_rn(ey, r2.y, __fmul_rn(ez, r2.z)));
  s.q0[slot] = r0;
  s.q1[slot] = r1;
  s.q2[slot] = make_float4(r2.x, r2.y, r2.z, den0);
  s.q3[slot] = make_float4(pu0, pv0, r3.w, r4.w);
}

struct CompArgs {
  SensorDev sd;
  Header* hdr;
  const unsigned int* tile_ranges;
  const double* beams;
  const float4* rec;
  float4* part;
  const unsigned int* vals;
  float4* pix;            // 2 x float4 per pixel: {D, A, Nx, Ny}, {Nz, last_pos, ncontrib, T_final}
  float* out_range; float* out_alpha; float* out_normal;
  const float* gD; const float* gA; const float* gN;
};

__global__ void __launch_bounds__(kCompThreads) composite_fwd_kernel(const CompArgs a) {
  __shared__ Stage st;
  __shared__ unsigned int s_contrib;
  const SensorDev& S = a.sd;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int tile = blockIdx.x;
  const TileGeom g = tile_geom(tile, S, a.beams, warp, lane);
  const unsigned int start = a.tile_ranges[2 * tile], end = a.tile_ranges[2 * tile + 1];
  if (tid == 0) s_contrib = 0;

  bool done = !g.inside;
  bool warp_done = __all_sync(0xffffffffu, done);
  float T = 1.f, D = 0.f, A = 0.f, Nx = 0.f, Ny = 0.f, Nz = 0.f;
  unsigned int ncontrib = 0, last_pos = 0;

  for (unsigned int base = start; base < end; base += kBatch) {
    const int nb = (int)min((unsigned int)kBatch, end - base);
    if (tid < nb) stage_entry(st, tid, a.rec + kRecVec * (size_t)a.vals[base + tid], g);
    __syncthreads();
    if (!warp_done) {
      for (int chunk = 0; chunk < nb; chunk += 32) {
        const int j = chunk + lane;
        bool hit = false;
        if (j < nb) { const float4 r = st.q3[j]; hit = rect_hits(__float_as_uint(r.z), __float_as_uint(r.w), g, S.W); }
        unsigned int mask = __ballot_sync(0xffffffffu, hit);
        while (mask) {
          const int b = __ffs(mask) - 1;
          mask &= mask - 1;
          const int jj = chunk + b;
          const float4 q0 = st.q0[jj], q1 = st.q1[jj], q2 = st.q2[jj], q3 = st.q3[jj];
          PairEval e;
          if (!done && eval_pair(g.ex, g.ey, g.ez, q0, q1, q2, q3, e)) {
            const float test = __fmul_rn(T, __fsub_rn(1.0f, e.a));
            if (test < LGS_T_MIN) done = true;      // stop; this surfel is not applied
            else {
              const float w = __fmul_rn(T, e.a);
              D = __fmaf_rn(w, e.tau, D);
              A = __fadd_rn(A, w);
              Nx = __fmaf_rn(w, q0.x, Nx); Ny = __fmaf_rn(w, q0.y, Ny); Nz = __fmaf_rn(w, q0.z, Nz);
              T = test;
              ++ncontrib;
              last_pos = (base - start) + (unsigned int)jj + 1u;
            }
          }
        }
        if (__all_sync(0xffffffffu, done)) { warp_done = true; break; }
      }
    }
    if (__syncthreads_and(warp_done)) break;
  }

  if (g.inside) {
    const size_t px = (size_t)g.row * S.W + g.col, HW = (size_t)S.H * S.W;
    a.out_range[px] = D;
    a.out_alpha[px] = A;
    if (a.out_normal) { a.out_normal[px] = Nx; a.out_normal[HW + px] = Ny; a.out_normal[2 * HW + px] = Nz; }
    a.pix[2 * px] = make_float4(D, A, Nx, Ny);
    a.pix[2 * px + 1] = make_float4(Nz, __uint_as_float(last_pos), __uint_as_float(ncontrib), T);
  }
  // contributing-pair counter (the "intersections" of BASELINE.json's metric)
  unsigned int wsum = ncontrib;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) wsum += __shfl_xor_sync(0xffffffffu, wsum, o);
  __syncthreads();
  if (lane == 0 && wsum) atomicAdd(&s_contrib, wsum);
  __syncthreads();
  if (tid == 0 && s_contrib) atomicAdd(&a.hdr->n_contrib, (unsigned long long)s_contrib);
}

// -------------------------------------------------------------------------------------------
// Backward composite (step S7).  Back to front over the entries [0, last_pos) of each pixel,
// starting from the stored T_final: T_i = T_{i+1} / (1 - a_i), S_i = sum_{j>i} w_j x_j grows from
// the back, so mostly-hidden surfels keep full relative accuracy.  The cut-off decisions are
// re-taken by the same eval_pair as the forward (bit-identical), the stop by last_pos.
// Per pair the plain adjoint of (u, v, tau) is accumulated in the surfel's own frame, where every
// term is O(1) (no cancellation): with ubar, vbar and zeta = (taubar + hbar.d)/(d.n),
//   sum ubar, sum vbar, sum zeta              -> dL/dc     = -(Su/s0) t_u - (Sv/s1) t_v + Sz n
//   sum ubar u, ubar v, vbar u, vbar v        -> dL/dt_u, dL/dt_v, dL/ds0 = -Suu/s0, dL/ds1 = -Svv/s1
//   sum zeta u, zeta v                        -> dL/dn     = -s0 Szu t_u - s1 Szv t_v + sigma sum w gN
//   sum w gN (3), sum G abar                  -> normal output, opacity
// The 13 sums are reduced over the warp with a transposed butterfly (16 shuffles) and added to
// the per-surfel partial row with one coalesced red.global per (warp, surfel)  -- north_star (4).
// -------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(kCompThreads) composite_bwd_kernel(const CompArgs a) {
  __shared__ Stage st;
  __shared__ float4 s_q4[kBatch];          // per-surfel constants of the adjoint: (t_u.c)/s0, (t_v.c)/s1, 1/k^f
  __shared__ unsigned int s_id[kBatch];
  __shared__ unsigned int s_maxpos;
  const SensorDev& S = a.sd;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int tile = blockIdx.x;
  const TileGeom g = tile_geom(tile, S, a.beams, warp, lane);
  const unsigned int start = a.tile_ranges[2 * tile];
  if (tid == 0) s_maxpos = 0;
  __syncthreads();

  float gd = 0.f, ga = 0.f, gnx = 0.f, gny = 0.f, gnz = 0.f, T = 1.f;
  unsigned int my_last = 0;
  if (g.inside) {
    const size_t px = (size_t)g.row * S.W + g.col, HW = (size_t)S.H * S.W;
    const float4 p1 = a.pix[2 * px + 1];
    gd = a.gD ? a.gD[px] : 0.f;
    ga = a.gA ? a.gA[px] : 0.f;
    if (a.gN) { gnx = a.gN[px]; gny = a.gN[HW + px]; gnz = a.gN[2 * HW + px]; }
    const bool any = (gd != 0.f) || (ga != 0.f) || (gnx != 0.f) || (gny != 0.f) || (gnz != 0.f);
    my_last = any ? __float_as_uint(p1.y) : 0u;
    T = p1.w;
  }
  unsigned int wmax = my_last;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) wmax = max(wmax, __shfl_xor_sync(0xffffffffu, wmax, o));
  if (lane == 0 && wmax) atomicMax(&s_maxpos, wmax);
  __syncthreads();
  const unsigned int cta_last = s_maxpos;     // entries [0, cta_last) of this tile's list matter
  float Ssuf = 0.f;

  const int nbatch = (int)((cta_last + kBatch - 1) / kBatch);
  for (int bi = nbatch - 1; bi >= 0; --bi) {
    const unsigned int off = (unsigned int)bi * kBatch;
    const int nb = (int)min((unsigned int)kBatch, cta_last - off);
    if (tid < nb) {
      const unsigned int id = a.vals[start + off + tid];
      stage_entry(st, tid, a.rec + kRecVec * (size_t)id, g);
      s_q4[tid] = __ldg(a.rec + kRecVec * (size_t)id + 5);
      s_id[tid] = id;
    }
    __syncthreads();
    if (off < wmax) {
      const int nbw = (int)min((unsigned int)nb, wmax - off);
      for (int chunk = ((nbw - 1) >> 5) << 5; chunk >= 0; chunk -= 32) {
        const int j = chunk + lane;
        bool hit = false;
        if (j < nbw) { const float4 r = st.q3[j]; hit = rect_hits(__float_as_uint(r.z), __float_as_uint(r.w), g, S.W); }
        unsigned int mask = __ballot_sync(0xffffffffu, hit);
        while (mask) {
          const int b = 31 - __clz(mask);
          mask &= ~(1u << b);
          const int jj = chunk + b;
          const float4 q0 = st.q0[jj], q1 = st.q1[jj], q2 = st.q2[jj], q3 = st.q3[jj];
          PairEval e;
          float v[16];
#pragma unroll
          for (int k = 0; k < 16; ++k) v[k] = 0.f;
          bool contrib = false;
          if ((off + (unsigned int)jj) < my_last && eval_pair(g.ex, g.ey, g.ez, q0, q1, q2, q3, e)) {
            // every pair before last_pos that passes the cut-offs was applied by the forward
            contrib = true;
            const float iom = rcp_approx(__fsub_rn(1.0f, e.a));
            const float Ti = T * iom;                 // transmittance in front of this surfel
            const float w = Ti * e.a;
            const float x = gd * e.tau + ga + (gnx * q0.x + gny * q0.y + gnz * q0.z);
            float abar = Ti * x - Ssuf * iom;
            Ssuf = __fmaf_rn(w, x, Ssuf);
            T = Ti;
            if (e.clamped) abar = 0.f;
            const float taubar = w * gd;
            const float Gbar = q1.w * abar;
            const float ubar = -e.u * e.G * Gbar, vbar = -e.v * e.G * Gbar;
            // zeta = (dL/dtau_total) / (d.n): sensitivity to moving the plane along its normal.
            // (t_u.d)/(d.n) = (u s0 + t_u.c)/k, so only per-surfel constants are needed.
            const float4 q4 = s_q4[jj];
            const float zeta = taubar * e.inv + (ubar * (e.u + q4.x) + vbar * (e.v + q4.y)) * q4.z;
            v[0] = ubar; v[1] = vbar; v[2] = zeta;
            v[3] = ubar * e.u; v[4] = ubar * e.v; v[5] = vbar * e.u; v[6] = vbar * e.v;
            v[7] = zeta * e.u; v[8] = zeta * e.v;
            v[9] = w * gnx; v[10] = w * gny; v[11] = w * gnz;
            v[12] = e.G * abar;
          }
          if (__any_sync(0xffffffffu, contrib)) {
            // transposed butterfly: after the steps lane l holds the warp total of value (l >> 1)
#pragma unroll
            for (int half = 8, m = 16; half >= 1; half >>= 1, m >>= 1) {
              const bool upper = (lane & m) != 0;
#pragma unroll
              for (int k = 0; k < half; ++k) {
                const float send = upper ? v[k] : v[k + half];
                const float keep = upper ? v[k + half] : v[k];
                v[k] = keep + __shfl_xor_sync(0xffffffffu, send, m);
              }
            }
            v[0] += __shfl_xor_sync(0xffffffffu, v[0], 1);
            const int slot = lane >> 1;
            if ((lane & 1) == 0 && slot < 13)
              atomicAdd(reinterpret_cast<float*>(a.part) + (size_t)s_id[jj] * kPartFloats + slot, v[0]);
          }
        }
      }
    }
    __syncthreads();
  }
}

// -------------------------------------------------------------------------------------------
// K8: per-surfel chain rule from the local-frame partial sums to (mu, q, s, alpha)  (step S8).
//   c = R_ws^T (mu - t_ws), [t_u t_v n] = R_ws^T R(q^), q^ = q/|q|; h = tau d - c = u s0 t_u + v s1 t_v.
// -------------------------------------------------------------------------------------------
struct ChainArgs {
  const float* mean; const float* quat; const float* scale;
  long long N;
  SensorDev sd;
  const float4* rec;
  float4* part;
  float* g_mean; float* g_quat; float* g_scale; float* g_opacity;
  int accumulate;
  const Header* hdr;
};

__global__ void __launch_bounds__(256) chain_kernel(const ChainArgs a) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= a.N) return;
  float gm[3] = {0.f, 0.f, 0.f}, gq[4] = {0.f, 0.f, 0.f, 0.f}, gs[2] = {0.f, 0.f}, go = 0.f;
  const float4 r3 = a.rec[kRecVec * i + 3];
  const bool visible = (__float_as_uint(r3.w) >> 16) != 0u && a.hdr->overflow == 0u;
  if (visible) {
    const float4 p0 = a.part[4 * i], p1 = a.part[4 * i + 1], p2 = a.part[4 * i + 2], p3 = a.part[4 * i + 3];
    // hand the row back zeroed, so that a further backward on the same forward starts clean
    a.part[4 * i] = a.part[4 * i + 1] = a.part[4 * i + 2] = a.part[4 * i + 3] = make_float4(0.f, 0.f, 0.f, 0.f);
    const float sg = a.rec[kRecVec * i + 2].w;       // sigma = -sign(n.c)
    const float Su = p0.x, Sv = p0.y, Sz = sg * p0.z, Suu = p0.w, Suv = p1.x, Svu = p1.y, Svv = p1.z;
    const float Szu = sg * p1.w, Szv = sg * p2.x;
    const float gnf[3] = {sg * p2.y, sg * p2.z, sg * p2.w};
    go = p3.x;
    // recompute the frame (fp32 is ample: every partial sum is already well conditioned)
    const SensorDev& S = a.sd;
    const float R[9] = {(float)S.R[0], (float)S.R[1], (float)S.R[2], (float)S.R[3], (float)S.R[4],
                        (float)S.R[5], (float)S.R[6], (float)S.R[7], (float)S.R[8]};
    const float4 qf = reinterpret_cast<const float4*>(a.quat)[i];
    const float2 sf = reinterpret_cast<const float2*>(a.scale)[i];
    const float qn = sqrtf(qf.x * qf.x + qf.y * qf.y + qf.z * qf.z + qf.w * qf.w);
    const float iq = 1.f / qn;
    const float w = qf.x * iq, x = qf.y * iq, y = qf.z * iq, z = qf.w * iq;
    const float E0[3] = {1.f - 2.f * (y * y + z * z), 2.f * (x * y + w * z), 2.f * (x * z - w * y)};
    const float E1[3] = {2.f * (x * y - w * z), 1.f - 2.f * (x * x + z * z), 2.f * (y * z + w * x)};
    const float E2[3] = {2.f * (x * z + w * y), 2.f * (y * z - w * x), 1.f - 2.f * (x * x + y * y)};
    const float s0 = sf.x, s1 = sf.y, is0 = 1.f / sf.x, is1 = 1.f / sf.y;
    // world-frame adjoints of mu and of the columns of R(q^): R_ws [..] with [t_u t_v n] = R_ws^T E
    // collapses to combinations of the columns E0, E1, E2 themselves.
    const float cu = -Su * is0, cv = -Sv * is1;
    float m0[3], m1[3], m2[3];
#pragma unroll
    for (int k = 0; k < 3; ++k) {
      gm[k] = cu * E0[k] + cv * E1[k] + Sz * E2[k];
      m0[k] = Suu * E0[k] + Suv * (s1 * is0) * E1[k];
      m1[k] = Svu * (s0 * is1) * E0[k] + Svv * E1[k];
      const float gw = R[3 * k] * gnf[0] + R[3 * k + 1] * gnf[1] + R[3 * k + 2] * gnf[2];   // R_ws (sum w gN)
      m2[k] = -s0 * Szu * E0[k] - s1 * Szv * E1[k] + gw;
    }
    gs[0] = -Suu * is0;
    gs[1] = -Svv * is1;
    // dL/dq^ = sum_j m_j . d(e_j)/dq^, written column by column from e_j(w, x, y, z)
    float gh[4];
    gh[0] = 2.f * (m0[1] * z - m0[2] * y - m1[0] * z + m1[2] * x + m2[0] * y - m2[1] * x);
    gh[1] = 2.f * (m0[1] * y + m0[2] * z + m1[0] * y - 2.f * m1[1] * x + m1[2] * w + m2[0] * z - m2[1] * w - 2.f * m2[2] * x);
    gh[2] = 2.f * (-2.f * m0[0] * y + m0[1] * x - m0[2] * w + m1[0] * x + m1[2] * z + m2[0] * w + m2[1] * z - 2.f * m2[2] * y);
    gh[3] = 2.f * (-2.f * m0[0] * z + m0[1] * w + m0[2] * x - m1[0] * w - 2.f * m1[1] * z + m1[2] * y + m2[0] * x + m2[1] * y);
    const float qg = w * gh[0] + x * gh[1] + y * gh[2] + z * gh[3];
    gq[0] = (gh[0] - w * qg) * iq; gq[1] = (gh[1] - x * qg) * iq;
    gq[2] = (gh[2] - y * qg) * iq; gq[3] = (gh[3] - z * qg) * iq;
  }
  if (a.accumulate) {
    if (visible) {
      a.g_mean[3 * i] += gm[0]; a.g_mean[3 * i + 1] += gm[1]; a.g_mean[3 * i + 2] += gm[2];
      float4* q = reinterpret_cast<float4*>(a.g_quat) + i;
      float4 qv = *q; qv.x += gq[0]; qv.y += gq[1]; qv.z += gq[2]; qv.w += gq[3]; *q = qv;
      float2* s = reinterpret_cast<float2*>(a.g_scale) + i;
      float2 sv = *s; sv.x += gs[0]; sv.y += gs[1]; *s = sv;
      a.g_opacity[i] += go;
    }
  } else {
    a.g_mean[3 * i] = gm[0]; a.g_mean[3 * i + 1] = gm[1]; a.g_mean[3 * i + 2] = gm[2];
    reinterpret_cast<float4*>(a.g_quat)[i] = make_float4(gq[0], gq[1], gq[2], gq[3]);
    reinterpret_cast<float2*>(a.g_scale)[i] = make_float2(gs[0], gs[1]);
    a.g_opacity[i] = go;
  }
}

CompArgs make_args(const SensorDev& sd, const Layout& L, char* ws, const uint32_t* vals) {
  CompArgs a;
  a.sd = sd;
  a.hdr = reinterpret_cast<Header*>(ws + L.hdr);
  a.tile_ranges = reinterpret_cast<const unsigned int*>(ws + L.tile_ranges);
  a.beams = reinterpret_cast<const double*>(ws + L.beams);
  a.rec = reinterpret_cast<const float4*>(ws + L.rec);
  a.part = reinterpret_cast<float4*>(ws + L.part);
  a.vals = vals;
  a.pix = reinterpret_cast<float4*>(ws + L.pix);
  a.out_range = a.out_alpha = a.out_normal = nullptr;
  a.gD = a.gA = a.gN = nullptr;
  return a;
}

}  // namespace

cudaError_t launch_composite_fwd(const SensorDev& sd, const Layout& L, char* ws, const uint64_t*, const uint32_t* vals,
                                 float* out_range, float* out_alpha, float* out_normal, cudaStream_t st) {
  CompArgs a = make_args(sd, L, ws, vals);
  a.out_range = out_range; a.out_alpha = out_alpha; a.out_normal = out_normal;
  composite_fwd_kernel<<<sd.ntiles, kCompThreads, 0, st>>>(a);
  return cudaGetLastError();
}

cudaError_t launch_composite_bwd(const SensorDev& sd, const Layout& L, char* ws, const uint32_t* vals, const float* gD,
                                 const float* gA, const float* gN, cudaStream_t st) {
  CompArgs a = make_args(sd, L, ws, vals);
  a.gD = gD; a.gA = gA; a.gN = gN;
  composite_bwd_kernel<<<sd.ntiles, kCompThreads, 0, st>>>(a);
  return cudaGetLastError();
}

cudaError_t launch_chain(const lgs_gaussians& g, const SensorDev& sd, const Layout& L, char* ws, float* g_mean,
                         float* g_quat, float* g_scale, float* g_opacity, int accumulate, cudaStream_t st) {
  if (g.N <= 0) return cudaSuccess;
  ChainArgs a;
  a.mean = g.mean; a.quat = g.quat; a.scale = g.scale;
  a.N = g.N; a.sd = sd;
  a.rec = reinterpret_cast<const float4*>(ws + L.rec);
  a.part = reinterpret_cast<float4*>(ws + L.part);
  a.g_mean = g_mean; a.g_quat = g_quat; a.g_scale = g_scale; a.g_opacity = g_opacity;
  a.accumulate = accumulate;
  a.hdr = reinterpret_cast<const Header*>(ws + L.hdr);
  chain_kernel<<<(unsigned)((g.N + 255) / 256), 256, 0, st>>>(a);
  return cudaGetLastError();
}

}  // namespace lgs
