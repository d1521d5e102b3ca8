// K5 / K7 / K8: front-to-back compositing (forward), its adjoint (backward: every pixel walks its own applied
// entries, vector reds into per-surfel rows) and the per-surfel chain rule to (mu, q, s, alpha).
//
// Steps S5, S7, S8 of SURVEY.md 8(a); north_star (3), (4).  What is rendered: PAPER.md:47 / 127
// (D^, A^, N^); cut-offs and ordering: DESIGN.md readings R3-R7, R15, R17.
//
// Work decomposition: the sorted lists are per 8x4 tile (lane = pixel), one
// CTA per tile.  Every warp composites a different 32-entry CHUNK of the list at the same time.
// Alpha compositing is associative: a chunk is composited locally from T = 1, the chunk
// transmittances are exchanged through shared memory, and the chunk results are combined in
// list order.  The early stop (T (1 - a) < 1e-4) is decided exactly: the first chunk whose
// cumulative transmittance falls below the threshold is re-walked by the lanes concerned with the
// true incoming T, later chunks are discarded for those pixels.
//
// Pair evaluation: with the per-surfel record
//   n^f = sigma n, k^f = sigma (n.c) = -|n.c|, A_u = sigma (t_v x c)/s0, A_v = sigma (c x t_u)/s1,
// a beam d hits the surfel plane at tau = k^f/(d.n^f) with local coordinates
// u = (d.A_u)/(d.n^f), v = (d.A_v)/(d.n^f): three dot products and one reciprocal per pair.
// All arithmetic of a pair is written with explicit round-to-nearest intrinsics so that every walk
// of the forward and of the backward kernel takes bit-identical cut-off decisions.
#include "lgs_internal.cuh"

namespace lgs {
namespace {

constexpr int kCompThreads = 256;
constexpr int kWarps = kCompThreads / 32;
constexpr int kChunk = 32;                 // list entries one warp composites per round
constexpr int kRound = kWarps * kChunk;    // list entries consumed per round
#ifndef LGS_GROUP
#define LGS_GROUP 2
#endif
constexpr int kGroup = LGS_GROUP;          // chunks per backward work item

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

__device__ __forceinline__ void red_add_v4(float* p, float x, float y, float z, float w) {
  asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(p), "f"(x), "f"(y), "f"(z), "f"(w) : "memory");
}

struct PairEval {
  float inv, u, v, G, a, tau;
  bool clamped;
};

// Anchored pair evaluation.  The beam of a pixel is d_p = d_a + delta with d_a the sub-tile's
// anchor beam (kept as hi + lo floats) and delta small, exact to ~6e-9.  At staging time each
// list entry gets its values at the anchor beam,
//   den0 = d_a.n^f,  pu0 = (d_a - c^).A_u,  pv0 = (d_a - c^).A_v      (c^.A_u = c^.A_v = 0 exactly),
// with c^ = c/|c| also kept as hi + lo, so the large products |A| ~ r/s only ever multiply the
// small vectors (d_a - c^) and delta.  Per pair: three 3-term fma chains and one reciprocal.
// Returns true if the pair passes every per-pair cut-off (den, 3 sigma, alpha >= 1/255).
// Branch-free: on a failed test the outputs are finite-or-not garbage and must not be used.
__device__ __forceinline__ bool eval_pair(float ex, float ey, float ez, const float4& q0, const float4& q1,
                                          const float4& q2, const float4& q3, PairEval& e) {
  const float den = __fmaf_rn(ex, q0.x, __fmaf_rn(ey, q0.y, __fmaf_rn(ez, q0.z, q2.w)));
  const bool ok_den = den < -LGS_DEN_MIN;         // else grazing or back-facing beam (tau <= 0)
  e.inv = rcp_approx(den);
  const float pu = __fmaf_rn(ex, q1.x, __fmaf_rn(ey, q1.y, __fmaf_rn(ez, q1.z, q3.x)));
  const float pv = __fmaf_rn(ex, q2.x, __fmaf_rn(ey, q2.y, __fmaf_rn(ez, q2.z, q3.y)));
  e.u = __fmul_rn(pu, e.inv);
  e.v = __fmul_rn(pv, e.inv);
  const float rho2 = __fmaf_rn(e.u, e.u, __fmul_rn(e.v, e.v));
  const bool ok_rho = rho2 <= LGS_RHO2_MAX;
  e.G = ex2_approx(__fmul_rn(rho2, -0.72134752044448170368f));   // exp(-rho2/2)
  const float araw = __fmul_rn(q1.w, e.G);
  e.clamped = araw > LGS_ALPHA_MAX;
  e.a = e.clamped ? LGS_ALPHA_MAX : araw;
  e.tau = __fmul_rn(q0.w, e.inv);
  return ok_den && ok_rho && (e.a >= LGS_ALPHA_MIN);
}

// Geometry of one tile: lane = pixel (8 columns x 4 rows).
struct SubGeom {
  int col, row;
  bool inside;
  float ex, ey, ez;                     // delta = d_p - d_a
  float ahx, ahy, ahz, alx, aly, alz;   // anchor beam d_a = hi + lo
};

__device__ __forceinline__ void beam64(const double* tab, int W, int H, int row, int col, double* d) {
  const double cph = tab[col], sph = tab[W + col], cth = tab[2 * W + row], sth = tab[2 * W + H + row];
  d[0] = cth * cph; d[1] = cth * sph; d[2] = sth;
}

__device__ __forceinline__ SubGeom sub_geom(int tile, const SensorDev& S, const double* tab, int lane) {
  SubGeom g;
  const int tr = tile / S.ntc, tc = tile - tr * S.ntc;
  const int col0 = tc * kTileW, row0 = tr * kTileH;
  g.col = col0 + (lane % kTileW);
  g.row = row0 + (lane / kTileW);
  g.inside = g.col < S.W && g.row < S.H;
  double da[3], dp[3];
  beam64(tab, S.W, S.H, min(row0 + kTileH / 2, S.H - 1), min(col0 + kTileW / 2, S.W - 1), da);
  g.ahx = (float)da[0]; g.ahy = (float)da[1]; g.ahz = (float)da[2];
  g.alx = (float)(da[0] - (double)g.ahx); g.aly = (float)(da[1] - (double)g.ahy); g.alz = (float)(da[2] - (double)g.ahz);
  beam64(tab, S.W, S.H, min(g.row, S.H - 1), min(g.col, S.W - 1), dp);
  g.ex = (float)(dp[0] - da[0]); g.ey = (float)(dp[1] - da[1]); g.ez = (float)(dp[2] - da[2]);
  return g;
}

// Staged (shared-memory) form of one list entry: 4 x float4, read by broadcast.
//   q0 = n^f.xyz, k^f | q1 = A_u.xyz, alpha | q2 = A_v.xyz, den0 | q3 = pu0, pv0, -, -
struct Staged { float4 q0, q1, q2, q3; };

__device__ __forceinline__ Staged stage_entry(const float4* __restrict__ rec, const SubGeom& g) {
  const float4 r0 = __ldg(rec), r1 = __ldg(rec + 1), r2 = __ldg(rec + 2), r3 = __ldg(rec + 3), r4 = __ldg(rec + 4);
  // e = d_a - c^ in two-float arithmetic (the hi parts nearly cancel, the lo parts restore the bits)
  const float ex = __fadd_rn(__fsub_rn(g.ahx, r3.x), __fsub_rn(g.alx, r4.x));
  const float ey = __fadd_rn(__fsub_rn(g.ahy, r3.y), __fsub_rn(g.aly, r4.y));
  const float ez = __fadd_rn(__fsub_rn(g.ahz, r3.z), __fsub_rn(g.alz, r4.z));
  const float den0 = __fmaf_rn(g.ahx, r0.x, __fmaf_rn(g.ahy, r0.y, __fmul_rn(g.ahz, r0.z)));
  const float pu0 = __fmaf_rn(ex, r1.x, __fmaf_rn(ey, r1.y, __fmul_rn(ez, r1.z)));
  const float pv0 = __fmaf_rn(ex, r2.x, __fmaf_rn(ey, r2.y, __fmul_rn(ez, r2.z)));
  Staged s;
  s.q0 = r0;
  s.q1 = r1;
  s.q2 = make_float4(r2.x, r2.y, r2.z, den0);
  s.q3 = make_float4(pu0, pv0, 0.f, 0.f);
  return s;
}

// Per-chunk summaries written by the forward for the backward: chunk c of a tile
// is its list entries [32 c, 32 c + 32).  Tiles lie back to back in the key array, so
// ((start + 32 c) >> 5) + tile is a distinct slot for every (tile, chunk).  Rows of a slot, one float
// per pixel (lane): 0 T behind the chunk, 1..5 the chunk's share of (D, A, Nx, Ny, Nz).
constexpr int kSumRows = 6;
__device__ __forceinline__ size_t chunk_slot(unsigned int start, unsigned int c, int tile) {
  return (size_t)((start + 32u * c) >> 5) + (size_t)tile;
}

struct CompArgs {
  SensorDev sd;
  Header* hdr;
  const unsigned int* tile_ranges;
  const uint4* tile_order;          // schedule {tile, start, end, -}, longest list first
  const double* beams;
  const float4* rec;
  float4* part;
  const unsigned int* vals;         // sorted values: surfel ids
  float2* pix;                      // per pixel: {last_pos (bits), T_final}
  float* sums;                      // per (tile, chunk) slot: [kSumRows][32] floats, see chunk_slot()
  unsigned int* pmask;              // per (tile, chunk) slot and pixel: bit j set iff the pixel may have applied entry j of the chunk
  uint4* tasks;                     // backward work items {tile, group of kGroup chunks, list start, list length}, listed by the forward
  float4* pixgeo;                   // per pixel: delta = d_p - d_a (written by the forward, read by the backward)
  float4* anchor;                   // per tile: anchor beam d_a as hi, lo (2 x float4)
  float* out_range; float* out_alpha; float* out_normal;
  const float* gD; const float* gA; const float* gN;
};

// -------------------------------------------------------------------------------------------
// Forward composite (step S5).
// -------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(kCompThreads, 3) composite_fwd_kernel(const CompArgs a) {
  __shared__ float4 s_st[kWarps][4][kChunk];
  __shared__ float s_tt[2][kWarps][32];        // chunk transmittances (double-buffered by round)
  __shared__ float s_tfin[32];                 // T at the stop, written by the warp that found it
  const SensorDev& S = a.sd;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  // Kernels that follow in the stream with programmatic stream serialisation and do not depend on this grid's output
  // (the loss stage's count kernel, the backward's clear kernel) may run beside its last wave.
  asm volatile("griddepcontrol.launch_dependents;");
  const uint4 sched = a.tile_order[blockIdx.x];
  const int tile = (int)sched.x;                               // global tile id: frame * ntiles_f + tile of the frame
  const int frame = (S.F == 1) ? 0 : tile / S.ntiles_f, tile_f = tile - frame * S.ntiles_f;
  const SubGeom g = sub_geom(tile_f, S, a.beams, lane);
  const unsigned int start = sched.y, len = sched.z - sched.y;
  const float4* __restrict__ rec_f = a.rec + kRecVec * (size_t)frame * (size_t)S.N;     // the frame's records

  bool done = !g.inside;             // identical in every warp (decided from shared data only)
  float Tc = 1.f;                    // transmittance carried into the current round (uniform over warps)
  float D = 0.f, A = 0.f, Nx = 0.f, Ny = 0.f, Nz = 0.f;   // this warp's share of the pixel sums
  unsigned int ncontrib = 0, last_pos = 0;
  unsigned int head = 0;
  int buf = 0;
  // the surfel id of this lane's entry is fetched one round ahead (one L2 round trip less per round)
  unsigned int id_next = 0;
  if ((unsigned int)(kChunk * warp + lane) < len) id_next = __ldg(a.vals + start + (unsigned int)(kChunk * warp + lane));

  while (head < len) {
    const int nthis = (int)min(len - head, (unsigned int)kRound);
    const int cnt = max(0, min(kChunk, nthis - kChunk * warp));
    const unsigned int slot0 = head + (unsigned int)(kChunk * warp);     // list position of this warp's chunk
    const unsigned int id = id_next;
    if (slot0 + (unsigned int)kRound + (unsigned int)lane < len) id_next = __ldg(a.vals + start + slot0 + (unsigned int)kRound + lane);
    if (lane < cnt) {
      const Staged s = stage_entry(rec_f + kRecVec * (size_t)id, g);
      s_st[warp][0][lane] = s.q0; s_st[warp][1][lane] = s.q1; s_st[warp][2][lane] = s.q2; s_st[warp][3][lane] = s.q3;
    }
    __syncwarp();
    // ---- speculative local walk of this warp's chunk, from T = 1 ---------------------------
    float t = 1.f, Dl = 0.f, Al = 0.f, Nxl = 0.f, Nyl = 0.f, Nzl = 0.f, tstop = 1.f;
    bool lstop = false;
    unsigned int amine = 0u, bit = 1u;           // entries of the chunk this lane applied (bit j = entry j)
#pragma unroll 4
    for (int j = 0; j < cnt; ++j, bit <<= 1) {
      const float4 q0 = s_st[warp][0][j], q1 = s_st[warp][1][j], q2 = s_st[warp][2][j], q3 = s_st[warp][3][j];
      PairEval e;
      const bool valid = eval_pair(g.ex, g.ey, g.ez, q0, q1, q2, q3, e);
      const float test = __fmul_rn(t, __fsub_rn(1.0f, e.a));
      const bool live = valid && !lstop;
      const bool stops = live && (test < LGS_T_MIN);
      const bool apply = live && !stops;
      if (stops) { lstop = true; tstop = test; }
      const float w = apply ? __fmul_rn(t, e.a) : 0.f;
      const float tau = apply ? e.tau : 0.f;
      Dl = __fmaf_rn(w, tau, Dl);
      Al = __fadd_rn(Al, w);
      Nxl = __fmaf_rn(w, q0.x, Nxl); Nyl = __fmaf_rn(w, q0.y, Nyl); Nzl = __fmaf_rn(w, q0.z, Nzl);
      if (apply) { t = test; amine |= bit; }
    }
    const int lastj = 31 - __clz(amine);         // -1 if none
    const unsigned int ncl = (unsigned int)__popc(amine);
    s_tt[buf][warp][lane] = lstop ? tstop : t;
    __syncthreads();
    // ---- combine in list order: incoming T of my chunk, first chunk that stops the pixel -----
    float Tb = Tc, Tmine = Tc;
    int kstop = kWarps;
#pragma unroll
    for (int k = 0; k < kWarps; ++k) {
      if (k == warp) Tmine = Tb;
      const float Tn = __fmul_rn(Tb, s_tt[buf][k][lane]);
      if (kstop == kWarps && Tn < LGS_T_MIN) kstop = k;
      Tb = (kstop == kWarps) ? Tn : Tb;
    }
    // Per (chunk, pixel) mask for the backward: the entries this pixel applied in the local walk from T = 1 -- a
    // superset of what the true incoming T allows (the backward cuts it at the pixel's last applied position);
    // pixels that stopped before this chunk hold 0.  One coalesced 128-byte row per chunk.
    if (cnt > 0) a.pmask[chunk_slot(start, slot0 >> 5, tile) * 32 + lane] = (done || warp > kstop) ? 0u : amine;
    if (!done && cnt > 0 && warp <= kstop) {
      float Tout, Dc, Ac, Nxc, Nyc, Nzc;
      if (warp < kstop) {
        Tout = __fmul_rn(Tmine, t);
        Dc = __fmul_rn(Tmine, Dl); Ac = __fmul_rn(Tmine, Al);
        Nxc = __fmul_rn(Tmine, Nxl); Nyc = __fmul_rn(Tmine, Nyl); Nzc = __fmul_rn(Tmine, Nzl);
        ncontrib += ncl;
        if (lastj >= 0) last_pos = slot0 + (unsigned int)lastj + 1u;
      } else {
        // the stop lies in this chunk: walk it again with the true incoming transmittance
        float T = Tmine;
        Dc = 0.f; Ac = 0.f; Nxc = 0.f; Nyc = 0.f; Nzc = 0.f;
        for (int j = 0; j < cnt; ++j) {
          const float4 q0 = s_st[warp][0][j], q1 = s_st[warp][1][j], q2 = s_st[warp][2][j], q3 = s_st[warp][3][j];
          PairEval e;
          if (eval_pair(g.ex, g.ey, g.ez, q0, q1, q2, q3, e)) {
            const float test = __fmul_rn(T, __fsub_rn(1.0f, e.a));
            if (test < LGS_T_MIN) break;            // stop; this surfel is not applied
            const float w = __fmul_rn(T, e.a);
            Dc = __fmaf_rn(w, e.tau, Dc);
            Ac = __fadd_rn(Ac, w);
            Nxc = __fmaf_rn(w, q0.x, Nxc); Nyc = __fmaf_rn(w, q0.y, Nyc); Nzc = __fmaf_rn(w, q0.z, Nzc);
            T = test;
            ++ncontrib;
            last_pos = slot0 + (unsigned int)j + 1u;
          }
        }
        // (no stop found: T is within rounding of the threshold and any further entry would stop)
        s_tfin[lane] = T;
        Tout = T;
      }
      D += Dc; A += Ac; Nx += Nxc; Ny += Nyc; Nz += Nzc;
      // chunk summary for the backward
      float* sm = a.sums + chunk_slot(start, slot0 >> 5, tile) * (kSumRows * 32) + lane;
      sm[0] = Tout; sm[32] = Dc; sm[64] = Ac; sm[96] = Nxc; sm[128] = Nyc; sm[160] = Nzc;
    }
    if (kstop < kWarps) done = true;
    Tc = Tb;
    head += (unsigned int)nthis;
    buf ^= 1;
    if (__all_sync(0xffffffffu, done)) break;     // same outcome in every warp
    // No barrier needed here: s_st is private to the warp and s_tt is double-buffered.
  }

  // ---- reduce the 8 warps' shares ----------------------------------------------------------------
  __syncthreads();
  float* red = reinterpret_cast<float*>(&s_st[0][0][0]);     // [7][kWarps][32]
  red[(0 * kWarps + warp) * 32 + lane] = D;
  red[(1 * kWarps + warp) * 32 + lane] = A;
  red[(2 * kWarps + warp) * 32 + lane] = Nx;
  red[(3 * kWarps + warp) * 32 + lane] = Ny;
  red[(4 * kWarps + warp) * 32 + lane] = Nz;
  red[(5 * kWarps + warp) * 32 + lane] = __uint_as_float(ncontrib);
  red[(6 * kWarps + warp) * 32 + lane] = __uint_as_float(last_pos);
  __syncthreads();
  if (warp == 0) {
    float d = 0.f, al = 0.f, nx = 0.f, ny = 0.f, nz = 0.f;
    unsigned int nc = 0, lp = 0;
#pragma unroll
    for (int w = 0; w < kWarps; ++w) {
      d += red[(0 * kWarps + w) * 32 + lane]; al += red[(1 * kWarps + w) * 32 + lane];
      nx += red[(2 * kWarps + w) * 32 + lane]; ny += red[(3 * kWarps + w) * 32 + lane];
      nz += red[(4 * kWarps + w) * 32 + lane];
      nc += __float_as_uint(red[(5 * kWarps + w) * 32 + lane]);
      lp = max(lp, __float_as_uint(red[(6 * kWarps + w) * 32 + lane]));
    }
    if (g.inside) {
      const size_t px = (size_t)g.row * S.W + g.col, HW = (size_t)S.H * S.W, fo = (size_t)frame * HW;
      a.out_range[fo + px] = d;
      a.out_alpha[fo + px] = al;
      if (a.out_normal) {
        float* on = a.out_normal + 3 * fo;
        on[px] = nx; on[HW + px] = ny; on[2 * HW + px] = nz;
      }
      a.pix[fo + px] = make_float2(__uint_as_float(lp), done ? s_tfin[lane] : Tc);
      if (frame == 0) a.pixgeo[px] = make_float4(g.ex, g.ey, g.ez, 0.f);       // (the frames share the grid)
    } else {
      nc = 0; lp = 0;
    }
    if (lane == 0 && frame == 0) {
      a.anchor[2 * tile_f] = make_float4(g.ahx, g.ahy, g.ahz, 0.f);
      a.anchor[2 * tile_f + 1] = make_float4(g.alx, g.aly, g.alz, 0.f);
    }
    // backward work items: one per group of kGroup chunks that reaches a pixel's last applied entry
    unsigned int top = lp;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) top = max(top, __shfl_xor_sync(0xffffffffu, top, o));
    const unsigned int ngr = (((top + 31u) >> 5) + (unsigned int)kGroup - 1u) / (unsigned int)kGroup;
    if (ngr) {
      unsigned int base = 0;
      if (lane == 0) base = atomicAdd(&a.hdr->n_tasks, ngr);
      base = __shfl_sync(0xffffffffu, base, 0);
      for (unsigned int c = lane; c < ngr; c += 32) a.tasks[base + c] = make_uint4((unsigned int)tile, c, start, len);
    }
    // contributing-pair counter (the "intersections" of BASELINE.json's metric)
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) nc += __shfl_xor_sync(0xffffffffu, nc, o);
    if (lane == 0 && nc) atomicAdd(&a.hdr->n_contrib, (unsigned long long)nc);
  }
}

// -------------------------------------------------------------------------------------------
// Backward composite (step S7).  One warp per work item (kGroup consecutive chunks of one tile's list; the items were
// listed by the forward), lane = pixel.  Every lane walks its own applied entries of a chunk
// back to front from the forward's exact T behind the chunk: T_i = T_{i+1} / (1 - a_i),
// S_i = sum_{j>i} w_j x_j grows from the back, so mostly-hidden surfels keep full relative
// accuracy.  The part of S that lies behind the chunk is the sum over the later chunks c' of
// gD D_c' + gA A_c' + gN.N_c' (the forward's chunk summaries), added from the back.  The cut-off
// decisions are re-taken by the same eval_pair as the forward (bit-identical), the stop by
// last_pos.  Chunks are independent: no barrier, no inter-warp exchange, and a long list spreads
// over the whole machine.
// Per pair the plain adjoint of (u, v, tau) is accumulated in the surfel's own frame, where every
// term is O(1) (no cancellation): with ubar, vbar and zeta = (taubar + hbar.d)/(d.n),
//   sum ubar, sum vbar, sum zeta              -> dL/dc     = -(Su/s0) t_u - (Sv/s1) t_v + Sz n
//   sum ubar u, ubar v, vbar u, vbar v        -> dL/dt_u, dL/dt_v, dL/ds0 = -Suu/s0, dL/ds1 = -Svv/s1
//   sum zeta u, zeta v                        -> dL/dn     = -s0 Szu t_u - s1 Szv t_v + sigma sum w gN
//   sum w gN (3), sum G abar                  -> normal output, opacity
// north_star (4) asks for a warp-shuffle reduction before the global atomics.  That form (a transposed butterfly, 17
// shuffles for the 13 sums, one red.global row per (warp, surfel)) was the first implementation; it walks every entry some
// pixel of the tile applied with all 32 lanes (~18 of a chunk's 32 entries at ~3.8 useful lanes).  The committed form walks
// per lane only the entries THAT pixel applied (~3.4 per chunk), so the lanes of a warp sit at different surfels and there
// is nothing to shuffle together; each pair adds its 13 sums with three red.global.add.v4.f32 and one scalar red (L2
// atomics; measured 2.6x the row rate of 13 scalar reds).  78 -> 65 us on config 2.
// -------------------------------------------------------------------------------------------
struct PixUp { float gd, ga, gnx, gny, gnz, Tfin; unsigned int last; };

// Upstream gradients and forward state of this lane's pixel; last = 0 if the pixel carries no gradient.
__device__ __forceinline__ PixUp load_pixel(const CompArgs& a, const SubGeom& g, int frame) {
  PixUp p;
  p.gd = p.ga = p.gnx = p.gny = p.gnz = 0.f; p.Tfin = 1.f; p.last = 0u;
  if (g.inside) {
    const size_t HW = (size_t)a.sd.H * a.sd.W, px = (size_t)g.row * a.sd.W + g.col, fo = (size_t)frame * HW;
    const float2 f = a.pix[fo + px];
    p.gd = a.gD ? a.gD[fo + px] : 0.f;
    p.ga = a.gA ? a.gA[fo + px] : 0.f;
    if (a.gN) { const float* gn = a.gN + 3 * fo; p.gnx = gn[px]; p.gny = gn[HW + px]; p.gnz = gn[2 * HW + px]; }
    const bool any = (p.gd != 0.f) || (p.ga != 0.f) || (p.gnx != 0.f) || (p.gny != 0.f) || (p.gnz != 0.f);
    p.last = any ? __float_as_uint(f.x) : 0u;
    p.Tfin = f.y;
  }
  return p;
}

#ifndef LGS_BWD_THREADS
#define LGS_BWD_THREADS 32
#endif
constexpr int kBwdThreads = LGS_BWD_THREADS;
constexpr int kBwdWarps = kBwdThreads / 32;

// Backward composite (step S7).  One warp per work item = up to kGroup consecutive chunks of one tile's list, walked
// back to front; lane = pixel.  Every lane walks ITS OWN applied entries of a chunk (the forward's per-pixel mask cut at
// the pixel's last applied position: on average ~3 of the chunk's 32 entries, against ~18 applied by some pixel of the
// tile), re-evaluates the pair bit-identically to the forward and runs the transmittance recurrence
// T_i = T_{i+1} / (1 - a_i), S_i = sum_{j>i} w_j x_j from the forward's exact T behind the chunk.  The lanes of a warp
// are then at different entries, so there is no warp reduction: each pair adds its 13 sums to the surfel's 64-byte row
// with red.global.add.v4.f32.
__global__ void __launch_bounds__(kBwdThreads, 1024 / kBwdThreads) composite_bwd_kernel(const CompArgs a) {
  __shared__ float4 s_st[kBwdWarps][5][kChunk];   // q0..q3 + adjoint constants (t_u.c)/s0, (t_v.c)/s1, 1/k^f
  __shared__ unsigned int s_id[kBwdWarps][kChunk];
  const SensorDev& S = a.sd;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  asm volatile("griddepcontrol.launch_dependents;");     // the chain kernel's CTAs come in as this grid drains, and wait
  const unsigned int ntasks = a.hdr->n_tasks;
  // One work item per warp, no pop counter (a shared counter would be thousands of atomics on ONE address, which the
  // L2 serialises: measured 17 % of the kernel's stall samples).  The grid covers the largest possible item count;
  // the hardware's block scheduler hands CTAs to SMs as warps retire, which balances items of very different cost.
  unsigned int task = blockIdx.x * kBwdWarps + warp;
  if (task >= ntasks) return;
  task = ntasks - 1u - task;          // heaviest first: the forward's CTAs of the longest tiles finish, and append, last
  const uint4 tk = a.tasks[task];
  const int tile = (int)tk.x;                                  // global tile id
  const int frame = (S.F == 1) ? 0 : tile / S.ntiles_f, tile_f = tile - frame * S.ntiles_f;
  const unsigned int start = tk.z, len = tk.w;
  const size_t row_f = (size_t)frame * (size_t)S.N;            // first per-(frame, surfel) row of the frame
  const int c_lo = kGroup * (int)tk.y;                       // the item's chunks: [c_lo, c_hi]
  const int c_hi = min(c_lo + kGroup - 1, (int)((len + 31u) >> 5) - 1);
  // geometry of the tile as the forward left it (anchor beam hi + lo per tile, delta beam per pixel)
  SubGeom g;
  {
    const int tr = tile_f / S.ntc, tc = tile_f - tr * S.ntc;
    g.col = tc * kTileW + (lane % kTileW);
    g.row = tr * kTileH + (lane / kTileW);
    g.inside = g.col < S.W && g.row < S.H;
    const float4 ah = __ldg(a.anchor + 2 * tile_f), al = __ldg(a.anchor + 2 * tile_f + 1);
    g.ahx = ah.x; g.ahy = ah.y; g.ahz = ah.z; g.alx = al.x; g.aly = al.y; g.alz = al.z;
    float4 e = make_float4(0.f, 0.f, 0.f, 0.f);
    if (g.inside) e = __ldg(a.pixgeo + (size_t)g.row * S.W + g.col);
    g.ex = e.x; g.ey = e.y; g.ez = e.z;
  }
  const PixUp p = load_pixel(a, g, frame);
  // per chunk of the item: this pixel's applied entries (the forward's local-walk mask cut at the pixel's last
  // applied position) and the forward's exact T behind the chunk -- all loads of the item issued together
  unsigned int mk[kGroup];
  float Tb[kGroup];
#pragma unroll
  for (int k = 0; k < kGroup; ++k) {
    const int c = c_lo + k;
    mk[k] = 0u; Tb[k] = 1.f;
    if (c <= c_hi && 32u * (unsigned int)c < p.last) {
      const size_t slot = chunk_slot(start, (unsigned int)c, tile);
      mk[k] = __ldg(a.pmask + slot * 32 + lane);
      Tb[k] = __ldg(a.sums + slot * (kSumRows * 32) + lane);
      const unsigned int nleft = p.last - 32u * (unsigned int)c;
      if (nleft < 32u) mk[k] &= (1u << nleft) - 1u;
    }
  }
  // S behind the item: the later chunks' shares of (D, A, N) against this pixel's upstream gradients, from the back
  float Ssuf = 0.f;
  if (p.last > 32u * (unsigned int)(c_hi + 1)) {
    const int clast = (int)((p.last - 1u) >> 5);
    for (int c1 = clast; c1 > c_hi; c1 -= 4) {
      float sc[4];
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        sc[k] = 0.f;
        const int c2 = c1 - k;
        if (c2 > c_hi) {
          const float* __restrict__ s2 = a.sums + chunk_slot(start, (unsigned int)c2, tile) * (kSumRows * 32) + lane;
          const float Dc = __ldg(s2 + 32), Ac = __ldg(s2 + 64), Nxc = __ldg(s2 + 96), Nyc = __ldg(s2 + 128), Nzc = __ldg(s2 + 160);
          sc[k] = __fmaf_rn(p.gd, Dc, __fmul_rn(p.ga, Ac)) + (p.gnx * Nxc + p.gny * Nyc + p.gnz * Nzc);
        }
      }
      Ssuf += sc[0]; Ssuf += sc[1]; Ssuf += sc[2]; Ssuf += sc[3];
    }
  }
#pragma unroll
  for (int k = kGroup - 1; k >= 0; --k) {                    // the item's chunks, back to front; S carries over
    unsigned int mine = mk[k];
    const unsigned int emask = __reduce_or_sync(0xffffffffu, mine);     // entries applied to some pixel
    if (emask == 0u) continue;                               // (warp-uniform)
    const unsigned int first = 32u * (unsigned int)(c_lo + k);          // list position of chunk entry 0
    float T = Tb[k];
    __syncwarp();                                            // the previous chunk's reads of s_st are done
    if ((emask >> lane) & 1u) {
      const unsigned int id = __ldg(a.vals + start + first + (unsigned int)lane);
      const float4* rec = a.rec + kRecVec * (row_f + (size_t)id);
      const Staged s = stage_entry(rec, g);
      s_st[warp][0][lane] = s.q0; s_st[warp][1][lane] = s.q1; s_st[warp][2][lane] = s.q2; s_st[warp][3][lane] = s.q3;
      s_st[warp][4][lane] = __ldg(rec + 5);
      s_id[warp][lane] = id;
    }
    __syncwarp();
    while (__any_sync(0xffffffffu, mine != 0u)) {
      if (mine != 0u) {
        const int j = 31 - __clz(mine);
        mine &= ~(1u << j);
        const float4 q0 = s_st[warp][0][j], q1 = s_st[warp][1][j], q2 = s_st[warp][2][j], q3 = s_st[warp][3][j];
        PairEval e;
        // (bit-identical to the forward's evaluation, so this is true for every bit of the mask; a false here
        // would mean a mismatch between the two walks and must not corrupt the chain)
        if (eval_pair(g.ex, g.ey, g.ez, q0, q1, q2, q3, e)) {
          const float iom = rcp_approx(__fsub_rn(1.0f, e.a));
          const float Ti = T * iom;                 // transmittance in front of this surfel
          const float w = Ti * e.a;
          const float x = __fmaf_rn(p.gd, e.tau, p.ga) + (p.gnx * q0.x + p.gny * q0.y + p.gnz * q0.z);
          float abar = Ti * x - Ssuf * iom;
          Ssuf = __fmaf_rn(w, x, Ssuf);
          T = Ti;
          if (e.clamped) abar = 0.f;
          const float taubar = w * p.gd;
          const float Gbar = q1.w * abar;
          const float ubar = -e.u * e.G * Gbar, vbar = -e.v * e.G * Gbar;
          // zeta = (dL/dtau_total) / (d.n): sensitivity to moving the plane along its normal.
          // (t_u.d)/(d.n) = (u s0 + t_u.c)/k, so only per-surfel constants are needed.
          const float4 q4 = s_st[warp][4][j];
          const float zeta = taubar * e.inv + (ubar * (e.u + q4.x) + vbar * (e.v + q4.y)) * q4.z;
          float* row = reinterpret_cast<float*>(a.part) + (row_f + (size_t)s_id[warp][j]) * kPartFloats;
          red_add_v4(row, ubar, vbar, zeta, ubar * e.u);
          red_add_v4(row + 4, ubar * e.v, vbar * e.u, vbar * e.v, zeta * e.u);
          red_add_v4(row + 8, zeta * e.v, w * p.gnx, w * p.gny, w * p.gnz);
          atomicAdd(row + 12, e.G * abar);
        }
      }
    }
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
  PoseSet poses;
  const uint4* emit;
  const float4* rec;
  const float4* part;
  float* g_mean; float* g_quat; float* g_scale; float* g_opacity;
  int accumulate;
  const Header* hdr;
};

// One thread per surfel; the frames of a batched call are added in frame order (the sum of the per-frame losses,
// DESIGN.md R18), exactly as F single-frame calls with accumulate = 1 would.
__global__ void __launch_bounds__(256) chain_kernel(const ChainArgs a) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  asm volatile("griddepcontrol.wait;" ::: "memory");      // launched beside the backward composite: wait for its sums
  if (i >= a.N) return;
  float gm[3] = {0.f, 0.f, 0.f}, gq[4] = {0.f, 0.f, 0.f, 0.f}, gs[2] = {0.f, 0.f}, go = 0.f;
  const float4 qf = reinterpret_cast<const float4*>(a.quat)[i];
  const float2 sf = reinterpret_cast<const float2*>(a.scale)[i];
  const bool ok = a.hdr->overflow == 0u;
  bool any = false;
  // the frame R(q^) = [E0 E1 E2] in the world (fp32 is ample: every partial sum is already well conditioned)
  const float qn = sqrtf(qf.x * qf.x + qf.y * qf.y + qf.z * qf.z + qf.w * qf.w);
  const float iq = 1.f / qn;
  const float w = qf.x * iq, x = qf.y * iq, y = qf.z * iq, z = qf.w * iq;
  const float E0[3] = {1.f - 2.f * (y * y + z * z), 2.f * (x * y + w * z), 2.f * (x * z - w * y)};
  const float E1[3] = {2.f * (x * y - w * z), 1.f - 2.f * (x * x + z * z), 2.f * (y * z + w * x)};
  const float E2[3] = {2.f * (x * z + w * y), 2.f * (y * z - w * x), 1.f - 2.f * (x * x + y * y)};
  const float s0 = sf.x, s1 = sf.y, is0 = 1.f / sf.x, is1 = 1.f / sf.y;
  const int nf = a.sd.F;
  for (int f = 0; f < nf; ++f) {
    const size_t r = (size_t)f * (size_t)a.N + (size_t)i;
    // every load is issued up front (one round trip): the rows of culled surfels are not used
    const uint4 em = a.emit[r];
    const float4 p0 = a.part[4 * r], p1 = a.part[4 * r + 1], p2 = a.part[4 * r + 2], p3 = a.part[4 * r + 3];
    const bool visible = (em.x >> 16) != 0u && ok;
    if (!visible) continue;
    any = true;
    const float sg = (em.w >> 31) ? -1.f : 1.f;      // sigma = -sign(n.c)
    const float Su = p0.x, Sv = p0.y, Sz = sg * p0.z, Suu = p0.w, Suv = p1.x, Svu = p1.y, Svv = p1.z;
    const float Szu = sg * p1.w, Szv = sg * p2.x;
    const float gnf[3] = {sg * p2.y, sg * p2.z, sg * p2.w};
    const double* Rd = a.poses.R[f];
    const float R[9] = {(float)Rd[0], (float)Rd[1], (float)Rd[2], (float)Rd[3], (float)Rd[4],
                        (float)Rd[5], (float)Rd[6], (float)Rd[7], (float)Rd[8]};
    // world-frame adjoints of mu and of the columns of R(q^): R_ws [..] with [t_u t_v n] = R_ws^T E
    // collapses to combinations of the columns E0, E1, E2 themselves.
    const float cu = -Su * is0, cv = -Sv * is1;
    float fm[3], m0[3], m1[3], m2[3];
#pragma unroll
    for (int k = 0; k < 3; ++k) {
      fm[k] = cu * E0[k] + cv * E1[k] + Sz * E2[k];
      m0[k] = Suu * E0[k] + Suv * (s1 * is0) * E1[k];
      m1[k] = Svu * (s0 * is1) * E0[k] + Svv * E1[k];
      const float gw = R[3 * k] * gnf[0] + R[3 * k + 1] * gnf[1] + R[3 * k + 2] * gnf[2];   // R_ws (sum w gN)
      m2[k] = -s0 * Szu * E0[k] - s1 * Szv * E1[k] + gw;
    }
    // dL/dq^ = sum_j m_j . d(e_j)/dq^, written column by column from e_j(w, x, y, z)
    float gh[4];
    gh[0] = 2.f * (m0[1] * z - m0[2] * y - m1[0] * z + m1[2] * x + m2[0] * y - m2[1] * x);
    gh[1] = 2.f * (m0[1] * y + m0[2] * z + m1[0] * y - 2.f * m1[1] * x + m1[2] * w + m2[0] * z - m2[1] * w - 2.f * m2[2] * x);
    gh[2] = 2.f * (-2.f * m0[0] * y + m0[1] * x - m0[2] * w + m1[0] * x + m1[2] * z + m2[0] * w + m2[1] * z - 2.f * m2[2] * y);
    gh[3] = 2.f * (-2.f * m0[0] * z + m0[1] * w + m0[2] * x - m1[0] * w - 2.f * m1[1] * z + m1[2] * y + m2[0] * x + m2[1] * y);
    const float qg = w * gh[0] + x * gh[1] + y * gh[2] + z * gh[3];
    // (frame 0 is assigned, the others are added: a single-frame call gives the same bits as before)
    if (f == 0) {
      gm[0] = fm[0]; gm[1] = fm[1]; gm[2] = fm[2];
      gs[0] = -Suu * is0; gs[1] = -Svv * is1; go = p3.x;
      gq[0] = (gh[0] - w * qg) * iq; gq[1] = (gh[1] - x * qg) * iq; gq[2] = (gh[2] - y * qg) * iq; gq[3] = (gh[3] - z * qg) * iq;
    } else {
      gm[0] += fm[0]; gm[1] += fm[1]; gm[2] += fm[2];
      gs[0] += -Suu * is0; gs[1] += -Svv * is1; go += p3.x;
      gq[0] += (gh[0] - w * qg) * iq; gq[1] += (gh[1] - x * qg) * iq; gq[2] += (gh[2] - y * qg) * iq; gq[3] += (gh[3] - z * qg) * iq;
    }
  }
  if (a.accumulate) {
    if (any) {
      a.g_mean[3 * i] += gm[0]; a.g_mean[3 * i + 1] += gm[1]; a.g_mean[3 * i + 2] += gm[2];
      float4* q = reinterpret_cast<float4*>(a.g_quat) + i;
      float4 qv = *q; qv.x += gq[0]; qv.y += gq[1]; qv.z += gq[2]; qv.w += gq[3]; *q = qv;
      float2* sp = reinterpret_cast<float2*>(a.g_scale) + i;
      float2 sv = *sp; sv.x += gs[0]; sv.y += gs[1]; *sp = sv;
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
  a.tile_order = reinterpret_cast<const uint4*>(ws + L.tile_order);
  a.beams = reinterpret_cast<const double*>(ws + L.beams);
  a.rec = reinterpret_cast<const float4*>(ws + L.rec);
  a.part = reinterpret_cast<float4*>(ws + L.part);
  a.vals = vals;
  a.pix = reinterpret_cast<float2*>(ws + L.pix);
  a.sums = reinterpret_cast<float*>(ws + L.sums);
  a.pmask = reinterpret_cast<unsigned int*>(ws + L.pmask);
  a.tasks = reinterpret_cast<uint4*>(ws + L.tasks);
  a.pixgeo = reinterpret_cast<float4*>(ws + L.pixgeo);
  a.anchor = reinterpret_cast<float4*>(ws + L.anchor);
  a.out_range = a.out_alpha = a.out_normal = nullptr;
  a.gD = a.gA = a.gN = nullptr;
  return a;
}

}  // namespace

cudaError_t launch_composite_fwd(const SensorDev& sd, const Layout& L, char* ws, const uint32_t* vals,
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
  const size_t max_items = L.nslots / kGroup + (size_t)sd.ntiles + 1;     // (as sized in make_layout)
  composite_bwd_kernel<<<(unsigned)((max_items + kBwdWarps - 1) / kBwdWarps), kBwdThreads, 0, st>>>(a);
  return cudaGetLastError();
}

cudaError_t launch_chain(const lgs_gaussians& g, const SensorDev& sd, const PoseSet& poses, const Layout& L, char* ws,
                         float* g_mean, float* g_quat, float* g_scale, float* g_opacity, int accumulate, cudaStream_t st) {
  if (g.N <= 0) return cudaSuccess;
  ChainArgs a;
  a.mean = g.mean; a.quat = g.quat; a.scale = g.scale;
  a.N = g.N; a.sd = sd; a.poses = poses;
  a.emit = reinterpret_cast<const uint4*>(ws + L.emit);
  a.rec = reinterpret_cast<const float4*>(ws + L.rec);
  a.part = reinterpret_cast<const float4*>(ws + L.part);
  a.g_mean = g_mean; a.g_quat = g_quat; a.g_scale = g_scale; a.g_opacity = g_opacity;
  a.accumulate = accumulate;
  a.hdr = reinterpret_cast<const Header*>(ws + L.hdr);
  return launch_pdl(chain_kernel, dim3((unsigned)((g.N + 255) / 256)), dim3(256), 0, st, a);
}

namespace {
// Zeroes every partial-sum row (small maps).  Same launch rule as below.
__global__ void __launch_bounds__(256) clear_all_kernel(uint4* p, size_t n16) {
  const uint4 z = make_uint4(0u, 0u, 0u, 0u);
  for (size_t k = (size_t)blockIdx.x * blockDim.x + threadIdx.x; k < n16; k += (size_t)gridDim.x * blockDim.x) p[k] = z;
  asm volatile("griddepcontrol.wait;" ::: "memory");
}

// Zeroes the partial sums of the (frame, surfel) pairs the projection found visible (one 16-byte read per pair, one
// 64-byte row written per visible pair: on the large-map workload ~15 % of the rows).
__global__ void __launch_bounds__(256) clear_partials_kernel(const uint4* __restrict__ emit, uint4* part, size_t nrows) {
  const uint4 z = make_uint4(0u, 0u, 0u, 0u);
  // one thread per row, no loop: every thread has its one load in flight at once (a grid-stride loop of dependent
  // load -> branch -> store round trips measured 58 us on 4 M rows)
  const size_t k = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k < nrows && (__ldg(reinterpret_cast<const unsigned int*>(emit + k)) >> 16) != 0u) {
    part[4 * k] = z; part[4 * k + 1] = z; part[4 * k + 2] = z; part[4 * k + 3] = z;
  }
  // Launched with programmatic stream serialisation beside its predecessor (the loss gradient kernel or the forward
  // composite, both of which let their dependents in early): no CTA may retire before that predecessor has completed,
  // or the backward composite -- ordered only behind THIS grid -- could start on half-written upstream images / chunk
  // summaries.  Same rule as tile_sort_small_kernel.
  asm volatile("griddepcontrol.wait;" ::: "memory");
}
}  // namespace

cudaError_t launch_clear_partials(const SensorDev& sd, const Layout& L, char* ws, cudaStream_t st) {
  const size_t nrows = (size_t)(sd.N > 0 ? sd.N : 0) * (size_t)sd.F;
  // up to 2^20 rows (64 MB) the plain streaming clear is faster (4.9 against 7.4 us at 300k rows); beyond, most rows
  // belong to culled surfels and only the visible ones are written
  if (nrows <= ((size_t)1 << 20))
    return launch_pdl(clear_all_kernel, dim3((unsigned)(sm_count() * 4)), dim3(256), 0, st,
                      reinterpret_cast<uint4*>(ws + L.part), nrows * 4);
  return launch_pdl(clear_partials_kernel, dim3((unsigned)((nrows + 255) / 256)), dim3(256), 0, st,
                    reinterpret_cast<const uint4*>(ws + L.emit), reinterpret_cast<uint4*>(ws + L.part), nrows);
}

}  // namespace lgs
