// K1a / K1b / K1c: project / cull / rect + per-tile key slots (K1a), tile ranges (K1b), key
// placement bucketed by tile (K1c).
//
// Step S1 + S2 + S4 of SURVEY.md 8(a): the spherical projection pi_s of PAPER.md:47
// applied to each surfel of the map G = {(mu, q, s~, alpha)}.  The rect / key rule is
// fp64, every operation individually rounded
// (__dmul_rn / __dadd_rn / __fma_rn / __ddiv_rn / __dsqrt_rn are never contracted),
// so that keys and rects are bit-identical to the CPU list reference.
// K1a takes, for every (surfel, tile) pair, an index inside the tile's future segment from the
// tile's counter (one returning atomic per pair; one 128-byte line per tile: atomics on
// neighbouring words of a line serialise in L2) and appends the tuple (tile, index, range bits,
// surfel id) to an unordered list (one append per warp); K1b (one CTA) scans the counters into
// [start, end) tile ranges and builds the tile schedule; K1c streams the tuples and writes
// (range bits, surfel id) at tile start + index.  One atomic per pair in the whole front end.
// The order inside a segment is arbitrary: the per-tile sort orders by (range bits, surfel id).
#include <cstring>
#include "lgs_internal.cuh"

namespace lgs {
namespace {

constexpr double kPi = 3.14159265358979323846;
constexpr double kRectEps = 1e-9;

__device__ __forceinline__ double dmul(double a, double b) { return __dmul_rn(a, b); }
__device__ __forceinline__ double dadd(double a, double b) { return __dadd_rn(a, b); }
__device__ __forceinline__ double dsub(double a, double b) { return __dsub_rn(a, b); }
__device__ __forceinline__ double dfma(double a, double b, double c) { return __fma_rn(a, b, c); }
__device__ __forceinline__ double ddiv(double a, double b) { return __ddiv_rn(a, b); }
__device__ __forceinline__ double dsqr(double a) { return __dsqrt_rn(a); }

struct ProjArgs {
  const float* mean; const float* quat; const float* scale; const float* opacity;
  long long N;                 // surfels of the map
  SensorDev sd;
  PoseSet poses;               // (read by the projection only)
  Header* hdr;
  unsigned int* tile_ctr;    // per tile kTileStride words: [0] key count
  uint4* tuples;             // unordered (tile, index in tile, range bits, surfel id), cap entries
  unsigned int* tile_ranges;
  uint4* tile_order;       // schedule entries {tile, start, end, -}: one load gives a consumer CTA its list
  double* beams;
  uint4* emit;             // per surfel: col_min | ncols << 16, row_min | row_max << 16, range bits, tile count | sigma sign << 31
  float4* rec;
  uint2* kv;               // (range bits, surfel id) bucketed by tile, unsorted: the sort's input
  long long cap;
  int n_cta;
  int batch;                 // (frame, surfel) pairs per thread: 1 .. kProjBatch (make_layout)
};

// Tiles of a rect: rows [tr0, tr1], ntcs tile columns starting at tc0 (wrapping).
struct TileSpan { int tc0, ntcs, tr0, tr1; };
__device__ __forceinline__ TileSpan tile_span(int col_min, int ncols, int row_min, int row_max, int W, int ntc) {
  TileSpan t;
  t.tr0 = row_min / kTileH; t.tr1 = row_max / kTileH;
  t.tc0 = col_min / kTileW;
  if (ncols >= W) t.ntcs = ntc;
  else {
    const int last = col_min + ncols - 1;
    if (last < W) t.ntcs = last / kTileW - t.tc0 + 1;
    else t.ntcs = (ntc - t.tc0) + ((last - W) / kTileW + 1);
    if (t.ntcs > ntc) t.ntcs = ntc;
  }
  return t;
}

// Tile of pair j of a surfel whose rect spans tile rows tr0.. and ntcs tile columns from tc0 (wrapping).
__device__ __forceinline__ unsigned int pair_tile(unsigned int j, int tr0, int tc0, int ntcs, int ntc) {
  const int tr = tr0 + (int)(j / (unsigned int)ntcs);
  int tc = tc0 + (int)(j % (unsigned int)ntcs);
  if (tc >= ntc) tc -= ntc;
  return (unsigned int)(tr * ntc + tc);
}

#ifndef LGS_SLOT_DEPTH
#define LGS_SLOT_DEPTH 4
#endif
#ifndef LGS_PROJ_CTAS
#define LGS_PROJ_CTAS 8
#endif
constexpr int kProjBatch = 8;                   // most (frame, surfel) pairs per thread of the projection (a.batch of them)
constexpr int kSlotDepth = LGS_SLOT_DEPTH;      // slot atomics of a surfel's first pairs are issued before its record is computed

// kBatched = false: one pair per thread, no pre-cull (a.batch == 1).
template <bool kBatched>
__global__ void __launch_bounds__(kProjThreads, LGS_PROJ_CTAS) project_kernel(const ProjArgs a) {
  __shared__ unsigned int s_wcnt[kProjThreads / 32];
  __shared__ unsigned short s_list[kProjBatch * kProjThreads];
  const int tid = threadIdx.x;
  const SensorDev& S = a.sd;
  const long long gi0 = (long long)blockIdx.x * kProjThreads + tid;     // this thread's own (frame, surfel) pair
  // the one-CTA ranges kernel may become resident beside this grid (it waits for this grid's completion)
  asm volatile("griddepcontrol.launch_dependents;");

  // ---- beam tables (fp64 sincos; the compositing kernels round per tile) ---------------------------
  for (long long j = gi0; j < S.W; j += (long long)a.n_cta * kProjThreads) {
    const double phi = -kPi + ((double)j + 0.5) * S.dphi;
    a.beams[j] = cos(phi);
    a.beams[S.W + j] = sin(phi);
  }
  for (long long j = gi0; j < S.H; j += (long long)a.n_cta * kProjThreads) {
    const double th = S.elev_max - ((double)j + 0.5) * S.dth;
    a.beams[2 * S.W + j] = cos(th);
    a.beams[2 * S.W + S.H + j] = sin(th);
  }

  // ---- pre-cull (fp32, conservative) and compaction --------------------------------------------------------------
  // A CTA owns kProjBatch * kProjThreads consecutive (frame, surfel) pairs.  Pairs that the exact rule below certainly
  // culls -- opacity / scale tests (exact), centre range outside the gates or the whole 3-sigma rect outside the vertical
  // field of view by a margin that covers the fp32 error -- get their "not visible" record here; the others are listed
  // in shared memory and the fp64 projection runs over the list in full warps (on the large-map workload ~80 % of the
  // surfels lie beyond r_max).  A listed pair is decided again, exactly, below: the lists do not depend on this test.
  const long long base0 = (long long)blockIdx.x * (a.batch * kProjThreads);
  const long long total_pairs = (long long)S.F * a.N;
  unsigned int n_maybe = 0;            // (uniform over the CTA)
  if (!kBatched) {                     // one pair per thread, no pre-cull: nothing to pack
    const long long left = total_pairs - base0;
    n_maybe = (unsigned int)(left < (long long)kProjThreads ? (left > 0 ? left : 0) : (long long)kProjThreads);
  }
  for (int sb = 0; sb < (kBatched ? a.batch : 0); ++sb) {
    const long long g0 = base0 + (long long)sb * kProjThreads + tid;
    bool maybe = g0 < total_pairs;
    if (maybe) {
      const int f0 = (int)((unsigned int)g0 / (unsigned int)a.N);      // (F * N <= 2^28)
      const long long i0 = g0 - (long long)f0 * a.N;
      const float mx = a.mean[3 * i0], my = a.mean[3 * i0 + 1], mz = a.mean[3 * i0 + 2];
      const float2 sf = reinterpret_cast<const float2*>(a.scale)[i0];
      const float al = a.opacity[i0];
      maybe = !((double)al < 1.0 / 255.0) && (sf.x > 0.f) && (sf.y > 0.f);
      const double* Rd = a.poses.R[f0];
      // mu - t in fp64 (exact for fp32 mu and the fp32 t of lgs_sensor up to the one final rounding): the error of d is
      // relative to |d| itself, however far from the origin the map and the pose are (UTM-style coordinates)
      const float dx = (float)((double)mx - a.poses.t[f0][0]), dy = (float)((double)my - a.poses.t[f0][1]),
                  dz = (float)((double)mz - a.poses.t[f0][2]);
      const float cx = (float)Rd[0] * dx + (float)Rd[3] * dy + (float)Rd[6] * dz;
      const float cy = (float)Rd[1] * dx + (float)Rd[4] * dy + (float)Rd[7] * dz;
      const float cz = (float)Rd[2] * dx + (float)Rd[5] * dy + (float)Rd[8] * dz;
      const float rho = sqrtf(cx * cx + cy * cy), r = sqrtf(cx * cx + cy * cy + cz * cz);
      // (fp32 error of r: a few 1e-7 of r; the margins are 1e-4 relative + 1 mm.  NaN compares false: kept.)
      if (r > S.r_max * 1.0001f + 1e-3f) maybe = false;
      if (r < S.r_min * 0.9999f - 1e-3f) maybe = false;
      // Every point the rect rule bounds lies within q = 6.8 max(s) of the centre in the (rho, z) half-plane; that disc
      // lies wholly above the top (below the bottom) of the field of view iff its centre is farther than q from the
      // ray of elevation elev_max (elev_min) on that side.  Margin: 1e-3 r + 1 mm.
      const float q = 6.8f * fmaxf(sf.x, sf.y) + 1e-3f * r + 1e-3f;
      if (q < r) {
        if (cz * S.cos_emax - rho * S.sin_emax > q) maybe = false;
        if (rho * S.sin_emin - cz * S.cos_emin > q) maybe = false;
      }
      if (!maybe) a.emit[g0] = make_uint4(0u, 0u, 0u, 0u);
    }
    const unsigned int bal = __ballot_sync(0xffffffffu, maybe);
    if ((tid & 31) == 0) s_wcnt[tid >> 5] = (unsigned int)__popc(bal);
    __syncthreads();
    unsigned int before = 0, tot = 0;
#pragma unroll
    for (int k = 0; k < kProjThreads / 32; ++k) {
      if (k < (tid >> 5)) before += s_wcnt[k];
      tot += s_wcnt[k];
    }
    if (maybe) s_list[n_maybe + before + (unsigned int)__popc(bal & ((1u << (tid & 31)) - 1u))] = (unsigned short)(sb * kProjThreads + tid);
    n_maybe += tot;
    __syncthreads();
  }
  unsigned int nvis_cta = 0;
  for (unsigned int rbase = 0; rbase < (kBatched ? n_maybe : 1u); rbase += kProjThreads) {
  const bool active = rbase + (unsigned int)tid < n_maybe;
  const long long gi = base0 + (active ? (kBatched ? (long long)s_list[rbase + tid] : (long long)tid) : 0);   // (frame, surfel) pair f * N + i
  const int f = (active && S.F > 1) ? (int)((unsigned int)gi / (unsigned int)a.N) : 0;
  const long long i = gi - (long long)f * a.N;
  const unsigned int tile0 = (unsigned int)(f * S.ntiles_f);            // first tile id of frame f
  // ---- per-surfel projection -----------------------------------------------------
  unsigned int cnt = 0;
  int tc0 = 0, ntcs = 0, tr0 = 0, tr1 = -1;
  int col_min_r = 0, ncols_r = 0, row_min_r = 0, row_max_r = -1;
  unsigned int keybits = 0;
  bool sg_neg = false;
  unsigned int ix[kSlotDepth];     // index inside the tile's segment of the surfel's first kSlotDepth pairs
#pragma unroll
  for (int r = 0; r < kSlotDepth; ++r) ix[r] = 0u;
  if (active) {
    const double mx = a.mean[3 * i], my = a.mean[3 * i + 1], mz = a.mean[3 * i + 2];
    const float4 qf = reinterpret_cast<const float4*>(a.quat)[i];
    const float2 sf = reinterpret_cast<const float2*>(a.scale)[i];
    const double alpha = a.opacity[i];
    const double s0 = sf.x, s1 = sf.y;
    const double* R = a.poses.R[f];
    const double dx = dsub(mx, a.poses.t[f][0]), dy = dsub(my, a.poses.t[f][1]), dz = dsub(mz, a.poses.t[f][2]);
    const double cx = dfma(R[0], dx, dfma(R[3], dy, dmul(R[6], dz)));
    const double cy = dfma(R[1], dx, dfma(R[4], dy, dmul(R[7], dz)));
    const double cz = dfma(R[2], dx, dfma(R[5], dy, dmul(R[8], dz)));
    const double r = dsqr(dfma(cz, cz, dfma(cy, cy, dmul(cx, cx))));
    const float rkey = __double2float_rn(r);
    bool alive = true;
    if (alpha < 1.0 / 255.0) alive = false;
    if (rkey < S.r_min || rkey > S.r_max) alive = false;
    const double smax = fmax(s0, s1);
    if (r <= dmul(3.0, smax)) alive = false;
    if (!(s0 > 0.0) || !(s1 > 0.0)) alive = false;
    const double qw = qf.x, qx = qf.y, qy = qf.z, qz = qf.w;
    double qn = dsqr(dfma(qz, qz, dfma(qy, qy, dfma(qx, qx, dmul(qw, qw)))));
    if (!(qn > 0.0) || !isfinite(qn)) { alive = false; qn = 1.0; }
    if (!isfinite(r)) alive = false;
    if (alive) {
      const double w = ddiv(qw, qn), x = ddiv(qx, qn), y = ddiv(qy, qn), z = ddiv(qz, qn);
      const double xx = dmul(x, x), yy = dmul(y, y), zz = dmul(z, z);
      const double xy = dmul(x, y), xz = dmul(x, z), yz = dmul(y, z), wx = dmul(w, x), wy = dmul(w, y), wz = dmul(w, z);
      const double e0[3] = {dsub(1.0, dmul(2.0, dadd(yy, zz))), dmul(2.0, dadd(xy, wz)), dmul(2.0, dsub(xz, wy))};
      const double e1[3] = {dmul(2.0, dsub(xy, wz)), dsub(1.0, dmul(2.0, dadd(xx, zz))), dmul(2.0, dadd(yz, wx))};
      const double e2[3] = {dmul(2.0, dadd(xz, wy)), dmul(2.0, dsub(yz, wx)), dsub(1.0, dmul(2.0, dadd(xx, yy)))};
      double tu[3], tv[3], n[3];
#pragma unroll
      for (int c = 0; c < 3; ++c) {
        tu[c] = dfma(R[c], e0[0], dfma(R[3 + c], e0[1], dmul(R[6 + c], e0[2])));
        tv[c] = dfma(R[c], e1[0], dfma(R[3 + c], e1[1], dmul(R[6 + c], e1[2])));
        n[c] = dfma(R[c], e2[0], dfma(R[3 + c], e2[1], dmul(R[6 + c], e2[2])));
      }
      const double k = dadd(dadd(dmul(n[0], cx), dmul(n[1], cy)), dmul(n[2], cz));
      if (!isfinite(k)) alive = false;
      // ---- rect: conservative (azimuth, elevation) bounds of the 3-sigma ellipse -------
      const double k0 = dmul(3.0, s0), k1 = dmul(3.0, s1);
      const double a0 = dmul(k0, tu[0]), a1 = dmul(k0, tu[1]), a2 = dmul(k0, tu[2]);
      const double b0 = dmul(k1, tv[0]), b1 = dmul(k1, tv[1]), b2 = dmul(k1, tv[2]);
      const double rho = dsqr(dfma(cy, cy, dmul(cx, cx)));
      double erx = 1.0, ery = 0.0;
      if (rho > 0.0) { erx = ddiv(cx, rho); ery = ddiv(cy, rho); }
      const double ar = dfma(a1, ery, dmul(a0, erx)), br = dfma(b1, ery, dmul(b0, erx));
      const double at = dfma(a1, erx, -dmul(a0, ery)), bt = dfma(b1, erx, -dmul(b0, ery));
      const double hr = dsqr(dfma(br, br, dmul(ar, ar)));
      const double ht = dsqr(dfma(bt, bt, dmul(at, at)));
      const double hz = dsqr(dfma(b2, b2, dmul(a2, a2)));
      const double rho_lo = dsub(rho, hr), rho_out = dadd(rho, hr);
      const double rho_hi = dsqr(dfma(ht, ht, dmul(rho_out, rho_out)));
      const double z_lo = dsub(cz, hz), z_hi = dadd(cz, hz);
      int col_min = 0, ncols = 0;
      double th_lo, th_hi;
      if (rho_lo > 0.0) {
        const double half = dadd(atan(ddiv(ht, rho_lo)), kRectEps);
        const double phc = atan2(cy, cx);
        const double flo = ceil(dsub(ddiv(dadd(dsub(phc, half), kPi), S.dphi), 0.5));
        const double fhi = floor(dsub(ddiv(dadd(dadd(phc, half), kPi), S.dphi), 0.5));
        const double fn = dadd(dsub(fhi, flo), 1.0);
        if (!(fn >= 1.0)) alive = false;
        else if (fn >= (double)S.W) { col_min = 0; ncols = S.W; }
        else {
          const long long lo = (long long)flo;
          col_min = (int)(((lo % S.W) + S.W) % S.W);
          ncols = (int)fn;
        }
        th_lo = dsub(atan2(z_lo, z_lo < 0.0 ? rho_lo : rho_hi), kRectEps);
        th_hi = dadd(atan2(z_hi, z_hi > 0.0 ? rho_lo : rho_hi), kRectEps);
      } else {
        col_min = 0; ncols = S.W;
        th_lo = z_lo > 0.0 ? dsub(atan2(z_lo, rho_hi), kRectEps) : -0.5 * kPi;
        th_hi = z_hi < 0.0 ? dadd(atan2(z_hi, rho_hi), kRectEps) : 0.5 * kPi;
      }
      double frlo = ceil(dsub(ddiv(dsub(S.elev_max, th_hi), S.dth), 0.5));
      double frhi = floor(dsub(ddiv(dsub(S.elev_max, th_lo), S.dth), 0.5));
      if (frlo < 0.0) frlo = 0.0;
      if (frhi > (double)(S.H - 1)) frhi = (double)(S.H - 1);
      if (!(frhi >= frlo)) alive = false;
      if (alive) {
        const int row_min = (int)frlo, row_max = (int)frhi;
        col_min_r = col_min; ncols_r = ncols; row_min_r = row_min; row_max_r = row_max;
        const TileSpan ts = tile_span(col_min, ncols, row_min, row_max, S.W, S.ntc);
        tc0 = ts.tc0; ntcs = ts.ntcs; tr0 = ts.tr0; tr1 = ts.tr1;
        cnt = (unsigned int)((tr1 - tr0 + 1) * ntcs);
        keybits = __float_as_uint(rkey);
        // one slot per (surfel, tile) pair: a returning atomic on the tile's counter; the round trips of the first
        // kSlotDepth pairs overlap the record arithmetic below
#pragma unroll
        for (int r = 0; r < kSlotDepth; ++r)
          if ((unsigned int)r < cnt)
            ix[r] = atomicAdd(&a.tile_ctr[(size_t)(tile0 + pair_tile((unsigned int)r, tr0, tc0, ntcs, S.ntc)) * kTileStride], 1u);
        // ---- record for the compositing kernels (fp64 -> fp32 once) ----------------------
        // sigma = -sign(k): n^f = sigma n faces the sensor; k^f = sigma k = -|k|; the A vectors
        // take the same sign so that u, v, tau are unchanged.
        const double sg = (k > 0.0) ? -1.0 : 1.0;
        sg_neg = k > 0.0;
        // (the record is not part of the bit-exact rule: correctly rounded reciprocals instead of full divisions)
        const double rs0 = __drcp_rn(s0), rs1 = __drcp_rn(s1);
        const double is0 = sg * rs0, is1 = sg * rs1;
        const double Aux = (tv[1] * cz - tv[2] * cy) * is0, Auy = (tv[2] * cx - tv[0] * cz) * is0,
                     Auz = (tv[0] * cy - tv[1] * cx) * is0;
        const double Avx = (cy * tu[2] - cz * tu[1]) * is1, Avy = (cz * tu[0] - cx * tu[2]) * is1,
                     Avz = (cx * tu[1] - cy * tu[0]) * is1;
        const float alpha_rec = (k == 0.0) ? 0.0f : (float)alpha;   // a surfel seen exactly edge-on never contributes
        // unit centre direction as hi + lo floats (anchor of the pair evaluation)
        const double ir = __drcp_rn(r);
        const double chx = cx * ir, chy = cy * ir, chz = cz * ir;
        const float hx = (float)chx, hy = (float)chy, hz = (float)chz;
        float4* rec = a.rec + kRecVec * gi;
        rec[0] = make_float4((float)(sg * n[0]), (float)(sg * n[1]), (float)(sg * n[2]), (float)(sg * k));
        rec[1] = make_float4((float)Aux, (float)Auy, (float)Auz, alpha_rec);
        rec[2] = make_float4((float)Avx, (float)Avy, (float)Avz, (float)sg);
        rec[3] = make_float4(hx, hy, hz, __uint_as_float((unsigned)col_min | ((unsigned)ncols << 16)));
        rec[4] = make_float4((float)(chx - (double)hx), (float)(chy - (double)hy), (float)(chz - (double)hz),
                             __uint_as_float((unsigned)row_min | ((unsigned)row_max << 16)));
        // constants of the adjoint: (t_u.c)/s0, (t_v.c)/s1, 1/k^f
        const double tuc = tu[0] * cx + tu[1] * cy + tu[2] * cz, tvc = tv[0] * cx + tv[1] * cy + tv[2] * cz;
        rec[5] = make_float4((float)(tuc * rs0), (float)(tvc * rs1), (k == 0.0) ? 0.f : (float)__drcp_rn(sg * k), 0.f);
      }
    }
    // ncols = 0 marks "not visible" (K1b, K8 and the debug unpack read this, not the record)
    // (.w: tile count, top bit = sign bit of sigma, read by the chain kernel)
    a.emit[gi] = cnt ? make_uint4((unsigned)col_min_r | ((unsigned)ncols_r << 16), (unsigned)row_min_r | ((unsigned)row_max_r << 16),
                                 keybits, cnt | (sg_neg ? 0x80000000u : 0u))
                    : make_uint4(0u, 0u, 0u, 0u);
  }
  // ---- the tuples (tile, index, range bits, surfel id) go to an unordered list: one append per warp -----
  const int lane = tid & 31;
  unsigned int incl = cnt;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const unsigned int v = __shfl_up_sync(0xffffffffu, incl, o);
    if (lane >= o) incl += v;
  }
  const unsigned int wtotal = __shfl_sync(0xffffffffu, incl, 31);
  if (wtotal) {
    unsigned int wbase = 0;
    if (lane == 31) wbase = atomicAdd(&a.hdr->n_tuples, wtotal);
    wbase = __shfl_sync(0xffffffffu, wbase, 31);
    const unsigned int w = wbase + incl - cnt;
    const unsigned int id = (unsigned int)i;
#pragma unroll
    for (int r = 0; r < kSlotDepth; ++r)
      if ((unsigned int)r < cnt && (long long)(w + r) < a.cap)
        a.tuples[w + r] = make_uint4(tile0 + pair_tile((unsigned int)r, tr0, tc0, ntcs, S.ntc), ix[r], keybits, id);
    for (unsigned int j = kSlotDepth; j < cnt; ++j) {       // surfels covering more than kSlotDepth tiles
      const unsigned int tl = tile0 + pair_tile(j, tr0, tc0, ntcs, S.ntc);
      const unsigned int x = atomicAdd(&a.tile_ctr[(size_t)tl * kTileStride], 1u);
      if ((long long)(w + j) < a.cap) a.tuples[w + j] = make_uint4(tl, x, keybits, id);
    }
  }
  // visible-surfel count (lgs_query only): one reduction per CTA
  nvis_cta += (unsigned int)__syncthreads_count(cnt > 0);
  }      // rounds over the CTA's list
  if (tid == 0 && nvis_cta) atomicAdd(&a.hdr->n_visible, nvis_cta);
}

// -------------------------------------------------------------------------------------------
// K1b: tile ranges.  One CTA: exclusive scan of the per-tile key counts -> [start, end), the
// key total / overflow flag, and the tile schedule (longest list first) of the sort and
// compositing kernels.
// -------------------------------------------------------------------------------------------
constexpr int kRangeThreads = 1024;
constexpr int kRangeWarps = kRangeThreads / 32;

// Adds 1 to s_bucket[b] for every lane, one shared atomic per distinct bucket of the warp; returns the
// lane's slot (old counter value + rank among the lanes of the same bucket).  The tiles of a warp fall
// into a handful of length buckets, so plain per-lane atomics would serialise on a few addresses.
__device__ __forceinline__ unsigned int bucket_take(unsigned int* s_bucket, int b, bool active, int lane) {
  const unsigned int peers = __match_any_sync(0xffffffffu, active ? b : -1 - lane);
  const unsigned int below = __popc(peers & ((1u << lane) - 1u));
  unsigned int base = 0;
  if (active && below == 0) base = atomicAdd(&s_bucket[b], (unsigned int)__popc(peers));
  base = __shfl_sync(0xffffffffu, base, __ffs(peers) - 1);
  return base + below;
}

constexpr int kRangeCache = 8;     // batches of kRangeThreads tile counters kept in registers (8,192 tiles); more: re-read

__global__ void __launch_bounds__(kRangeThreads) ranges_kernel(const ProjArgs a) {
  __shared__ unsigned int s_warp_tot[kRangeWarps];
  __shared__ unsigned long long s_tot[kRangeWarps];
  __shared__ unsigned int s_bucket[34];
  __shared__ unsigned int s_ovf;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int ntiles = a.sd.ntiles;
  // Launched with programmatic stream serialisation: this CTA is resident while the projection still runs and
  // starts the moment it has completed; the placement kernel is let in now and waits for this one in turn.
  asm volatile("griddepcontrol.wait;" ::: "memory");
  asm volatile("griddepcontrol.launch_dependents;");
  if (tid < 34) s_bucket[tid] = 0;
  const int nb = (ntiles + kRangeThreads - 1) / kRangeThreads;
  // the counters of the first kRangeCache batches: one round trip, all loads in flight together
  unsigned int cc[kRangeCache];
#pragma unroll
  for (int b = 0; b < kRangeCache; ++b) {
    const int t = b * kRangeThreads + tid;
    cc[b] = (b < nb && t < ntiles) ? a.tile_ctr[(size_t)t * kTileStride] : 0u;
  }
  __syncthreads();
  // pass 0: key total (decides overflow before any range is published) and the length-bucket sizes
  unsigned long long tot64 = 0;
  auto pass0 = [&](unsigned int c, int t) {
    tot64 += c;
    bucket_take(s_bucket, 32 - __clz(c), t < ntiles, lane);       // bucket 0: empty list ... 32
  };
#pragma unroll
  for (int b = 0; b < kRangeCache; ++b)
    if (b < nb) pass0(cc[b], b * kRangeThreads + tid);
  for (int b = kRangeCache; b < nb; ++b) {
    const int t = b * kRangeThreads + tid;
    pass0((t < ntiles) ? a.tile_ctr[(size_t)t * kTileStride] : 0u, t);
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) tot64 += __shfl_xor_sync(0xffffffffu, tot64, o);
  if (lane == 0) s_tot[warp] = tot64;
  __syncthreads();
  if (warp == 0) {
    unsigned long long need = s_tot[lane];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) need += __shfl_xor_sync(0xffffffffu, need, o);
    const bool ovf = need > (unsigned long long)a.cap;
    if (lane == 0) {
      s_ovf = ovf ? 1u : 0u;
      a.hdr->n_keys_total = need;
      a.hdr->overflow = ovf ? 1u : 0u;
      a.hdr->n_keys = ovf ? 0u : (unsigned int)need;
    }
    // tiles ordered longest list first: counting sort on the bit length of the list length (the order
    // inside a bucket is irrelevant).  Bucket b starts after all longer buckets.  On overflow every list
    // is empty (bucket 0).
    unsigned int c0 = ovf ? 0u : s_bucket[32 - lane];    // lane l holds bucket 32 - l; bucket 0 comes last
    unsigned int inc = c0;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const unsigned int v = __shfl_up_sync(0xffffffffu, inc, o);
      if (lane >= o) inc += v;
    }
    __syncwarp();
    s_bucket[32 - lane] = inc - c0;
    if (lane == 31) s_bucket[0] = inc;
    if (32 - lane == kSortBigBucket - 1) a.hdr->n_big = inc - c0;      // tiles in buckets >= kSortBigBucket come first
  }
  __syncthreads();
  const bool ovf = s_ovf != 0u;
  unsigned int carry = 0;
  auto pass1 = [&](unsigned int c, int t) {
    unsigned int inc = c;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const unsigned int v = __shfl_up_sync(0xffffffffu, inc, o);
      if (lane >= o) inc += v;
    }
    __syncthreads();
    if (lane == 31) s_warp_tot[warp] = inc;
    __syncthreads();
    // exclusive offset of this warp and the batch total: warp scan of the 32 warp totals
    unsigned int wt = s_warp_tot[lane], winc = wt;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const unsigned int v = __shfl_up_sync(0xffffffffu, winc, o);
      if (lane >= o) winc += v;
    }
    const unsigned int woff = __shfl_sync(0xffffffffu, winc - wt, warp);
    const unsigned int tot = __shfl_sync(0xffffffffu, winc, 31);
    const unsigned int end = carry + woff + inc;
    const unsigned int slot = bucket_take(s_bucket, 32 - __clz(c), t < ntiles, lane);
    if (t < ntiles) {
      *reinterpret_cast<uint2*>(a.tile_ranges + 2 * t) = make_uint2(end - c, end);
      a.tile_order[slot] = make_uint4((unsigned int)t, end - c, end, 0u);
    }
    carry += tot;
  };
#pragma unroll
  for (int b = 0; b < kRangeCache; ++b)
    if (b < nb) pass1(ovf ? 0u : cc[b], b * kRangeThreads + tid);
  for (int b = kRangeCache; b < nb; ++b) {
    const int t = b * kRangeThreads + tid;
    pass1((t < ntiles && !ovf) ? a.tile_ctr[(size_t)t * kTileStride] : 0u, t);
  }
}

// -------------------------------------------------------------------------------------------
// K1c: key placement.  Streams the unordered tuples (tile, index, range bits, surfel id) of K1a and
// writes (range bits, surfel id) at tile start + index: no atomics, coalesced 16-byte reads.
// -------------------------------------------------------------------------------------------
constexpr int kPlaceThreads = 256;

__global__ void __launch_bounds__(kPlaceThreads) emit_kernel(const ProjArgs a) {
  asm volatile("griddepcontrol.wait;" ::: "memory");      // launched beside the ranges kernel: wait for its results
  if (a.hdr->overflow) return;                 // the frame renders as zeros; lgs_query reports the need
  const unsigned int n = a.hdr->n_keys;
  for (unsigned int k = blockIdx.x * kPlaceThreads + threadIdx.x; k < n; k += gridDim.x * kPlaceThreads) {
    const uint4 t = a.tuples[k];
    const unsigned int pos = __ldg(a.tile_ranges + 2 * t.x) + t.y;
    a.kv[pos] = make_uint2(t.z, t.w);          // one 8-byte store per key (the scattered stores bound this kernel)
  }
}

// Test-only: rects [N,4] from the emission records; keys64 / surfel ids of the sorted lists.
__global__ void unpack_rects_kernel(const uint4* emit, long long N, int4* out) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N) return;
  const uint4 e = emit[i];
  const int ncols = (int)(e.x >> 16);
  out[i] = ncols ? make_int4((int)(e.x & 0xffffu), ncols, (int)(e.y & 0xffffu), (int)(e.y >> 16)) : make_int4(0, 0, 0, 0);
}

__global__ void unpack_keys_kernel(const unsigned int* ranges, const unsigned int* keys, const unsigned int* vals,
                                   unsigned long long* keys_out, unsigned int* vals_out) {
  const unsigned int tile = blockIdx.x;
  const unsigned int s = ranges[2 * tile], e = ranges[2 * tile + 1];
  for (unsigned int p = s + threadIdx.x; p < e; p += blockDim.x) {
    if (keys_out) keys_out[p] = ((unsigned long long)tile << 32) | keys[p];
    if (vals_out) vals_out[p] = vals[p];
  }
}

ProjArgs make_proj_args(const lgs_gaussians& g, const SensorDev& sd, const Layout& L, char* ws) {
  ProjArgs a;
  memset(&a.poses, 0, sizeof(a.poses));
  a.mean = g.mean; a.quat = g.quat; a.scale = g.scale; a.opacity = g.opacity;
  a.N = g.N;
  a.sd = sd;
  a.hdr = reinterpret_cast<Header*>(ws + L.hdr);
  a.tile_ctr = reinterpret_cast<unsigned int*>(ws + L.tile_ctr);
  a.tuples = reinterpret_cast<uint4*>(ws + L.sums);     // dead before the forward composite writes its summaries
  a.tile_ranges = reinterpret_cast<unsigned int*>(ws + L.tile_ranges);
  a.tile_order = reinterpret_cast<uint4*>(ws + L.tile_order);
  a.beams = reinterpret_cast<double*>(ws + L.beams);
  a.emit = reinterpret_cast<uint4*>(ws + L.emit);
  a.rec = reinterpret_cast<float4*>(ws + L.rec);
  // the tuples take the first 16 bytes per key of the summaries' region, the placed pairs the next 8
  a.kv = reinterpret_cast<uint2*>(ws + L.sums + (size_t)L.cap * 16);
  a.cap = L.cap;
  a.n_cta = L.n_proj_cta;
  a.batch = L.proj_batch;
  return a;
}

}  // namespace

cudaError_t launch_project(const lgs_gaussians& g, const SensorDev& sd, const PoseSet& poses, const Layout& L, char* ws,
                           cudaStream_t st) {
  ProjArgs a = make_proj_args(g, sd, L, ws);
  a.poses = poses;
  if (a.batch > 1) project_kernel<true><<<L.n_proj_cta, kProjThreads, 0, st>>>(a);
  else project_kernel<false><<<L.n_proj_cta, kProjThreads, 0, st>>>(a);
  return cudaGetLastError();
}

cudaError_t launch_ranges(const SensorDev& sd, const Layout& L, char* ws, cudaStream_t st) {
  lgs_gaussians g;
  g.mean = g.quat = g.scale = g.opacity = nullptr;
  g.N = 0;
  return launch_pdl(ranges_kernel, dim3(1), dim3(kRangeThreads), 0, st, make_proj_args(g, sd, L, ws));
}

cudaError_t launch_emit(const lgs_gaussians& g, const SensorDev& sd, const Layout& L, char* ws, cudaStream_t st) {
  const long long want = (L.cap + kPlaceThreads - 1) / kPlaceThreads;
  // One key per thread (the loop of the kernel only runs once): every thread's two dependent loads are in flight at
  // once.  A grid of 8 CTAs per SM striding over the keys is a chain of ~120 dependent round trips per thread on the
  // 36 M keys of configs[4] (measured 652 us).
  const long long most = (long long)1 << 22;
  const unsigned grid = (unsigned)(want < most ? (want > 0 ? want : 1) : most);
  return launch_pdl(emit_kernel, dim3(grid), dim3(kPlaceThreads), 0, st, make_proj_args(g, sd, L, ws));
}

cudaError_t launch_unpack_lists(const SensorDev& sd, const Layout& L, const char* ws, int64_t N, uint64_t* keys_out,
                                uint32_t* vals_out, int32_t* rects_out, cudaStream_t st) {
  if (rects_out && N > 0)
    unpack_rects_kernel<<<(unsigned)((N + 255) / 256), 256, 0, st>>>(reinterpret_cast<const uint4*>(ws + L.emit), N,
                                                                   reinterpret_cast<int4*>(rects_out));
  if (keys_out || vals_out)
    unpack_keys_kernel<<<sd.ntiles, 256, 0, st>>>(reinterpret_cast<const unsigned int*>(ws + L.tile_ranges),
                                                  reinterpret_cast<const unsigned int*>(ws + L.keys0),
                                                  reinterpret_cast<const unsigned int*>(ws + L.vals0),
                                                  reinterpret_cast<unsigned long long*>(keys_out), vals_out);
  return cudaGetLastError();
}

}  // namespace lgs
