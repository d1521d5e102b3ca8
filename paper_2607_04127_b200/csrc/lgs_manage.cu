// K12-K15: map management (section 3.3 "Control Score", section 3.5 "Real-time Map
// Budget Control"): control score (Eq. 9), quantile Q_q, structure-aware
// adaptive split, one pass of planar cover-and-prune, keep-flag compaction.
// Readings R29-R36 of DESIGN.md section 3 fix what the paper leaves open (normalisation, quantile rule, caps, tie
// rules, children, cover region); every such constant is a caller input.  Decisions (candidate, cell, representative,
// inside / outside, ranks) are integer work taken in fp32 with explicitly rounded operations in a fixed order, the same
// order oracle/map_manage.py writes, so that flags and indices can be compared bit for bit.
// Building blocks: an exact k-th order statistic by radix select on the float bit patterns (four 8-bit passes, each a
// multi-CTA histogram + a one-warp pick; all state stays on the device), block counts + one-CTA scan + in-block ballot
// ranks for every order-preserving selection, and the per-tile segmented sort of lgs_sort.cu for the per-cell quantile.
#include "lgs_internal.cuh"

namespace lgs {
namespace {

constexpr int kMT = 256;                 // threads per block of the per-surfel kernels

// ---- control score -----------------------------------------------------------------------------------------------
struct ScoreArgs {
  long long N;
  const float* sigma; const float* res;
  float lo[3], inv[3], w[3], eps;        // inv = 1 / (hi - lo)
  float* c;
};

__global__ void __launch_bounds__(kMT) control_score_kernel(const ScoreArgs a) {
  const long long i = (long long)blockIdx.x * kMT + threadIdx.x;
  if (i >= a.N) return;
  const float s0 = a.sigma[3 * i], s1 = a.sigma[3 * i + 1], s2 = a.sigma[3 * i + 2];
  const float l0 = s0 * s0, l1 = s1 * s1, l2 = s2 * s2;                  // lambda_{i,j} = sigma_{i,j}^2
  const float x[3] = {(l0 - l1) / (l0 + a.eps), l2 / (l0 + l1 + l2 + a.eps), a.res[i]};
  float c = 0.f;
#pragma unroll
  for (int k = 0; k < 3; ++k) c += a.w[k] * fminf(fmaxf((x[k] - a.lo[k]) * a.inv[k], 0.f), 1.f);
  a.c[i] = fminf(fmaxf(c, 0.f), 1.f);
}

// ---- radix select: the k-th smallest (or largest) of the keys that satisfy a predicate ------------------------------
// Keys are the bit patterns of non-negative floats (ordered as unsigned integers).  State on the device:
struct SelectState {
  unsigned int prefix;       // bits decided so far (the digits of the passes done)
  unsigned int k;            // 1-based rank still to be found among the keys that match the prefix
  unsigned int count;        // number of keys taking part (filled by the count kernel)
  unsigned int found;        // 1 once the result is valid (0: no key takes part)
  unsigned int hist[4][256];
};

struct SelectArgs {
  long long N;
  const unsigned int* keys;          // float bits
  const float* thr;                  // optional predicate: key value (as float) > *thr ...
  const float* opacity; float alpha_min;   // ... and opacity >= alpha_min (split candidates); NULL: every key
  SelectState* st;
  int pass, descending;
  unsigned int cap;                  // k = min(cap, count) for the descending (split) use
  long long krank;                   // k for the ascending (quantile) use
  float* out;                        // result as float (device)
};

__device__ __forceinline__ bool select_pred(const SelectArgs& a, long long i, unsigned int key) {
  if (!a.thr) return true;
  return __uint_as_float(key) > *a.thr && a.opacity[i] >= a.alpha_min;
}

__global__ void __launch_bounds__(kMT) select_hist_kernel(const SelectArgs a) {
  __shared__ unsigned int s_h[256];
  s_h[threadIdx.x] = 0u;
  __syncthreads();
  const SelectState& S = *a.st;
  const int shift = 24 - 8 * a.pass;
  const unsigned int himask = a.pass == 0 ? 0u : (0xffffffffu << (shift + 8));
  const unsigned int prefix = S.prefix;
  for (long long i = (long long)blockIdx.x * kMT + threadIdx.x; i < a.N; i += (long long)gridDim.x * kMT) {
    const unsigned int key = a.keys[i];
    if ((key & himask) == prefix && select_pred(a, i, key)) atomicAdd(&s_h[(key >> shift) & 255u], 1u);
  }
  __syncthreads();
  if (s_h[threadIdx.x]) atomicAdd(&a.st->hist[a.pass][threadIdx.x], s_h[threadIdx.x]);
}

// One warp: walks the 256 digit counts from the bottom (ascending) or the top (descending) to the digit that holds
// rank k, fixes that digit in the prefix and reduces k by the keys passed over.
__global__ void select_pick_kernel(const SelectArgs a) {
  SelectState& S = *a.st;
  if (threadIdx.x != 0) return;
  if (a.pass == 0) {
    unsigned int n = 0;
    for (int d = 0; d < 256; ++d) n += S.hist[0][d];
    S.count = n;
    unsigned long long k = a.descending ? (unsigned long long)min(a.cap, n) : (unsigned long long)a.krank;
    if (k > n) k = n;
    S.k = (unsigned int)k;
    S.found = (n > 0 && k > 0) ? 1u : 0u;
  }
  if (S.found) {
    unsigned int k = S.k, acc = 0;
    const int shift = 24 - 8 * a.pass;
    for (int t = 0; t < 256; ++t) {
      const int d = a.descending ? 255 - t : t;
      const unsigned int h = S.hist[a.pass][d];
      if (acc + h >= k) { S.prefix |= (unsigned int)d << shift; S.k = k - acc; break; }
      acc += h;
    }
  }
  if (a.pass == 3 && a.out) *a.out = S.found ? __uint_as_float(S.prefix) : 0.f;
}

cudaError_t run_select(SelectArgs a, cudaStream_t st) {
  cudaError_t e = cudaMemsetAsync(a.st, 0, sizeof(SelectState), st);
  if (e != cudaSuccess) return e;
  const long long want = (a.N + kMT - 1) / kMT;
  const unsigned grid = (unsigned)max(1ll, min(want, (long long)sm_count() * 8));
  for (int p = 0; p < 4; ++p) {
    a.pass = p;
    select_hist_kernel<<<grid, kMT, 0, st>>>(a);
    select_pick_kernel<<<1, 32, 0, st>>>(a);
  }
  return cudaGetLastError();
}

// ---- block counts / scan / in-block rank: the order-preserving selection pattern ------------------------------------
// One-CTA exclusive scan of `nb` block counts (in place) + total; two interleaved sequences if blk2 != NULL.
__global__ void __launch_bounds__(1024) scan_blocks_kernel(unsigned int* blk, unsigned int* blk2, long long nb,
                                                          unsigned int* total, unsigned int* total2) {
  __shared__ unsigned int s_w[2][32];
  __shared__ unsigned int s_carry[2];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  if (tid < 2) s_carry[tid] = 0u;
  __syncthreads();
  for (long long base = 0; base < nb; base += 1024) {
    const long long b = base + tid;
    unsigned int c[2] = {(b < nb) ? blk[b] : 0u, (b < nb && blk2) ? blk2[b] : 0u};
    unsigned int inc[2] = {c[0], c[1]};
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
#pragma unroll
      for (int q = 0; q < 2; ++q) {
        const unsigned int v = __shfl_up_sync(0xffffffffu, inc[q], o);
        if (lane >= o) inc[q] += v;
      }
    }
    if (lane == 31) { s_w[0][warp] = inc[0]; s_w[1][warp] = inc[1]; }
    __syncthreads();
    unsigned int woff[2] = {0u, 0u}, tot[2] = {0u, 0u};
    for (int w = 0; w < 32; ++w)
      for (int q = 0; q < 2; ++q) { const unsigned int x = s_w[q][w]; if (w < warp) woff[q] += x; tot[q] += x; }
    const unsigned int carry[2] = {s_carry[0], s_carry[1]};
    if (b < nb) { blk[b] = carry[0] + woff[0] + inc[0] - c[0]; if (blk2) blk2[b] = carry[1] + woff[1] + inc[1] - c[1]; }
    __syncthreads();
    if (tid < 2) s_carry[tid] = carry[tid] + tot[tid];
    __syncthreads();
  }
  if (tid == 0) { if (total) *total = s_carry[0]; if (total2) *total2 = s_carry[1]; }
}

// rank of this thread among the threads of its block with pred (exclusive), and nothing else
__device__ __forceinline__ unsigned int block_rank(bool pred, unsigned int* s_w) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const unsigned int bal = __ballot_sync(0xffffffffu, pred);
  if (lane == 0) s_w[warp] = (unsigned int)__popc(bal);
  __syncthreads();
  unsigned int woff = 0;
#pragma unroll
  for (int w = 0; w < kMT / 32; ++w) woff += (w < warp) ? s_w[w] : 0u;
  __syncthreads();
  return woff + (unsigned int)__popc(bal & ((1u << lane) - 1u));
}

// ---- fp32 frame with explicitly rounded operations (same sequence as oracle/map_manage.py _frame_uv) -----------------
__device__ __forceinline__ void frame_uv(const float4 q, float* tu, float* tv) {
  const float n = __fsqrt_rn(__fadd_rn(__fadd_rn(__fadd_rn(__fmul_rn(q.x, q.x), __fmul_rn(q.y, q.y)), __fmul_rn(q.z, q.z)),
                                       __fmul_rn(q.w, q.w)));
  const float w = __fdiv_rn(q.x, n), x = __fdiv_rn(q.y, n), y = __fdiv_rn(q.z, n), z = __fdiv_rn(q.w, n);
  const float xx = __fmul_rn(x, x), yy = __fmul_rn(y, y), zz = __fmul_rn(z, z);
  const float xy = __fmul_rn(x, y), xz = __fmul_rn(x, z), yz = __fmul_rn(y, z);
  const float wx = __fmul_rn(w, x), wy = __fmul_rn(w, y), wz = __fmul_rn(w, z);
  tu[0] = __fsub_rn(1.f, __fmul_rn(2.f, __fadd_rn(yy, zz)));
  tu[1] = __fmul_rn(2.f, __fadd_rn(xy, wz));
  tu[2] = __fmul_rn(2.f, __fsub_rn(xz, wy));
  tv[0] = __fmul_rn(2.f, __fsub_rn(xy, wz));
  tv[1] = __fsub_rn(1.f, __fmul_rn(2.f, __fadd_rn(xx, zz)));
  tv[2] = __fmul_rn(2.f, __fadd_rn(yz, wx));
}

// ---- adaptive split (readings R31, R32) ----------------------------------------------------------------
struct SplitArgs {
  long long N;
  const float* c; const float* thr; float alpha_min;
  unsigned int cap;
  float shift, log_shrink;
  float* mean; float* quat; float* log_scale; float* opacity; float* scale; float* m; float* v;
  unsigned char* flags;            // [N] out (may be NULL): 1 = split
  long long* n_new;                // N + number of splits
  SelectState* st;
  unsigned int* blk_a; unsigned int* blk_b;     // per block counts / offsets
  unsigned int* tot;               // [0] candidates above the cut, [1] ties (unused), [2] splits
};

__device__ __forceinline__ bool split_cand(const SplitArgs& a, long long i, float ci) {
  return i < a.N && ci > *a.thr && a.opacity[i] >= a.alpha_min;
}

// per block: candidates strictly above the cut score t (the k-th largest candidate score), and candidates equal to it
__global__ void __launch_bounds__(kMT) split_count_kernel(const SplitArgs a) {
  const long long i = (long long)blockIdx.x * kMT + threadIdx.x;
  const float t = __uint_as_float(a.st->prefix);
  const float ci = i < a.N ? a.c[i] : 0.f;
  const bool cand = a.st->found && split_cand(a, i, ci);
  const unsigned int ngt = (unsigned int)__syncthreads_count(cand && ci > t);
  const unsigned int nti = (unsigned int)__syncthreads_count(cand && ci == t);
  if (threadIdx.x == 0) { a.blk_a[blockIdx.x] = nti; a.blk_b[blockIdx.x] = ngt; }
}

// decides the splits (ties at the cut score in index order), writes the flags and the per-block split counts
__global__ void __launch_bounds__(kMT) split_flag_kernel(const SplitArgs a, unsigned char* sel) {
  __shared__ unsigned int s_w[kMT / 32];
  const long long i = (long long)blockIdx.x * kMT + threadIdx.x;
  const float t = __uint_as_float(a.st->prefix);
  const float ci = i < a.N ? a.c[i] : 0.f;
  const bool cand = a.st->found && split_cand(a, i, ci);
  const unsigned int want = min(a.cap, a.st->count);               // k of the selection
  const unsigned int n_gt = a.tot[0];
  const bool tie = cand && ci == t;
  const unsigned int trank = a.blk_a[blockIdx.x] + block_rank(tie, s_w);
  const bool s = cand && (ci > t || (tie && n_gt + trank < want));
  if (i < a.N) sel[i] = s ? 1 : 0;
  const unsigned int ns = (unsigned int)__syncthreads_count(s);
  __syncthreads();
  if (threadIdx.x == 0) a.blk_b[blockIdx.x] = ns;
}

__global__ void __launch_bounds__(kMT) split_apply_kernel(const SplitArgs a, const unsigned char* sel) {
  __shared__ unsigned int s_w[kMT / 32];
  const long long i = (long long)blockIdx.x * kMT + threadIdx.x;
  const bool s = i < a.N && sel[i] != 0;
  const unsigned int r = a.blk_b[blockIdx.x] + block_rank(s, s_w);
  if (blockIdx.x == 0 && threadIdx.x == 0) *a.n_new = a.N + (long long)a.tot[2];
  if (!s) return;
  const long long j = a.N + (long long)r;                          // row of the appended child
  const float4 q = reinterpret_cast<const float4*>(a.quat)[i];
  float tu[3], tv[3];
  frame_uv(q, tu, tv);
  const float ls0 = a.log_scale[2 * i], ls1 = a.log_scale[2 * i + 1];
  const float d = a.shift * expf(ls0);                             // shift * s_{i,0} along a_i = R(q_i) e_0
  const float mx = a.mean[3 * i], my = a.mean[3 * i + 1], mz = a.mean[3 * i + 2];
  a.mean[3 * i] = mx + d * tu[0]; a.mean[3 * i + 1] = my + d * tu[1]; a.mean[3 * i + 2] = mz + d * tu[2];
  a.mean[3 * j] = mx - d * tu[0]; a.mean[3 * j + 1] = my - d * tu[1]; a.mean[3 * j + 2] = mz - d * tu[2];
  reinterpret_cast<float4*>(a.quat)[j] = q;
  const float c0 = ls0 - a.log_shrink, c1 = ls1 - a.log_shrink;
  a.log_scale[2 * i] = c0; a.log_scale[2 * i + 1] = c1; a.log_scale[2 * j] = c0; a.log_scale[2 * j + 1] = c1;
  a.opacity[j] = a.opacity[i];
  if (a.scale) {
    const float e0 = expf(c0), e1 = expf(c1);
    a.scale[2 * i] = e0; a.scale[2 * i + 1] = e1; a.scale[2 * j] = e0; a.scale[2 * j + 1] = e1;
  }
  for (int k = 0; k < 10; ++k) {
    if (a.m) { a.m[10 * i + k] = 0.f; a.m[10 * j + k] = 0.f; }
    if (a.v) { a.v[10 * i + k] = 0.f; a.v[10 * j + k] = 0.f; }
  }
}

}  // namespace

// workspace of lgs_quantile / lgs_split / lgs_compact: select state + two block-count arrays + totals + N flag bytes
size_t manage_workspace_bytes(int64_t N) {
  const size_t nb = (size_t)((N + kMT - 1) / kMT + 1);
  return align_up(sizeof(SelectState)) + 2 * align_up(nb * 4) + 256 + align_up((size_t)(N > 0 ? N : 1));
}

struct ManageWs {
  SelectState* st; unsigned int* blk_a; unsigned int* blk_b; unsigned int* tot; unsigned char* flags;
};
static ManageWs carve_manage(void* ws, int64_t N) {
  const size_t nb = (size_t)((N + kMT - 1) / kMT + 1);
  char* p = static_cast<char*>(ws);
  ManageWs w;
  w.st = reinterpret_cast<SelectState*>(p); p += align_up(sizeof(SelectState));
  w.blk_a = reinterpret_cast<unsigned int*>(p); p += align_up(nb * 4);
  w.blk_b = reinterpret_cast<unsigned int*>(p); p += align_up(nb * 4);
  w.tot = reinterpret_cast<unsigned int*>(p); p += 256;
  w.flags = reinterpret_cast<unsigned char*>(p);
  return w;
}

cudaError_t launch_control_score(int64_t N, const float* sigma, const float* res, const float* bounds, const float* w,
                                 float eps, float* c, cudaStream_t st) {
  if (N <= 0) return cudaSuccess;
  ScoreArgs a;
  a.N = N; a.sigma = sigma; a.res = res; a.eps = eps; a.c = c;
  for (int k = 0; k < 3; ++k) { a.lo[k] = bounds[2 * k]; a.inv[k] = 1.0f / (bounds[2 * k + 1] - bounds[2 * k]); a.w[k] = w[k]; }
  control_score_kernel<<<(unsigned)((N + kMT - 1) / kMT), kMT, 0, st>>>(a);
  return cudaGetLastError();
}

cudaError_t launch_quantile(int64_t N, const float* x, long long krank, float* out, void* workspace, cudaStream_t st) {
  SelectArgs a = {};
  a.N = N; a.keys = reinterpret_cast<const unsigned int*>(x); a.thr = nullptr; a.opacity = nullptr; a.alpha_min = 0.f;
  a.st = carve_manage(workspace, N).st; a.descending = 0; a.cap = 0; a.krank = krank; a.out = out;
  return run_select(a, st);
}

cudaError_t launch_split(int64_t N, const float* c, const float* thr, float alpha_min, unsigned int cap, float shift,
                         float shrink, float* mean, float* quat, float* log_scale, float* opacity, float* scale, float* m,
                         float* v, unsigned char* flags_out, long long* n_new, void* workspace, cudaStream_t st) {
  const ManageWs w = carve_manage(workspace, N);
  SelectArgs s = {};
  s.N = N; s.keys = reinterpret_cast<const unsigned int*>(c); s.thr = thr; s.opacity = opacity; s.alpha_min = alpha_min;
  s.st = w.st; s.descending = 1; s.cap = cap; s.krank = 0; s.out = nullptr;
  cudaError_t e = run_select(s, st);
  if (e != cudaSuccess) return e;
  SplitArgs a;
  a.N = N; a.c = c; a.thr = thr; a.alpha_min = alpha_min; a.cap = cap; a.shift = shift; a.log_shrink = logf(shrink);
  a.mean = mean; a.quat = quat; a.log_scale = log_scale; a.opacity = opacity; a.scale = scale; a.m = m; a.v = v;
  a.flags = flags_out; a.n_new = n_new; a.st = w.st; a.blk_a = w.blk_a; a.blk_b = w.blk_b; a.tot = w.tot;
  const long long nb = (N + kMT - 1) / kMT;
  unsigned char* sel = flags_out ? flags_out : w.flags;
  if (nb > 0) split_count_kernel<<<(unsigned)nb, kMT, 0, st>>>(a);
  scan_blocks_kernel<<<1, 1024, 0, st>>>(w.blk_a, w.blk_b, nb, w.tot + 1, w.tot);          // tie offsets; total above the cut
  if (nb > 0) split_flag_kernel<<<(unsigned)nb, kMT, 0, st>>>(a, sel);
  scan_blocks_kernel<<<1, 1024, 0, st>>>(w.blk_b, nullptr, nb, w.tot + 2, nullptr);        // split offsets; total
  split_apply_kernel<<<(unsigned)(nb > 0 ? nb : 1), kMT, 0, st>>>(a, sel);
  return cudaGetLastError();
}

// ---- planar cover-and-prune, one pass (readings R33-R36) -------------------------------------------
namespace {

struct CoverArgs {
  long long N;
  const float* mean; const float* quat; float* scale; float* log_scale; const float* opacity; const float* c;
  const float* thr;
  CoverParams P;
  long long ncell;
  int* cellid;                         // [N] cell of a planar candidate, -1 otherwise
  unsigned int* rho2;                  // [N] float bits of a member's rho^2
  unsigned long long* repkey;          // [ncell] max over candidates of alpha bits << 32 | ~index
  unsigned int* cnt; unsigned int* start; unsigned int* cursor; unsigned int* ranges; float* R2;
  unsigned int* keys0; unsigned int* vals0;
  unsigned int* blk; unsigned int* tot;
  unsigned char* keep; long long* n_removed;
};

__device__ __forceinline__ int cover_cell(const CoverArgs& a, long long i) {
  const float ma = a.mean[3 * i + a.P.axis_a], mb = a.mean[3 * i + a.P.axis_b];
  const float fa = floorf(__fdiv_rn(__fsub_rn(ma, a.P.origin_a), a.P.cell));
  const float fb = floorf(__fdiv_rn(__fsub_rn(mb, a.P.origin_b), a.P.cell));
  if (!(fa >= 0.f && fa < (float)a.P.dim_a && fb >= 0.f && fb < (float)a.P.dim_b)) return -1;     // (false for NaN)
  return (int)fa * a.P.dim_b + (int)fb;
}

__global__ void __launch_bounds__(kMT) cover_assign_kernel(const CoverArgs a) {
  const long long i = (long long)blockIdx.x * kMT + threadIdx.x;
  if (i >= a.N) return;
  int cell = -1;
  const float al = a.opacity[i];
  if (a.c[i] <= *a.thr && al >= a.P.alpha_min) cell = cover_cell(a, i);          // planar candidate inside the grid
  a.cellid[i] = cell;
  if (cell >= 0) {
    atomicMax(&a.repkey[cell], ((unsigned long long)__float_as_uint(al) << 32) | (unsigned long long)(0xffffffffu - (unsigned int)i));
    atomicAdd(&a.cnt[cell], 1u);
  }
}

__global__ void __launch_bounds__(kMT) cover_members_count_kernel(const CoverArgs a) {
  const long long g = (long long)blockIdx.x * kMT + threadIdx.x;
  if (g < a.ncell) { const unsigned int n = a.cnt[g]; a.start[g] = n ? n - 1u : 0u; }
}

__global__ void __launch_bounds__(kMT) cover_ranges_kernel(const CoverArgs a) {
  const long long g = (long long)blockIdx.x * kMT + threadIdx.x;
  if (g < a.ncell) {
    const unsigned int n = a.cnt[g], s = a.start[g];
    a.ranges[2 * g] = s; a.ranges[2 * g + 1] = s + (n ? n - 1u : 0u);
  }
}

__global__ void __launch_bounds__(kMT) cover_member_kernel(const CoverArgs a) {
  const long long i = (long long)blockIdx.x * kMT + threadIdx.x;
  if (i >= a.N) return;
  const int cell = a.cellid[i];
  if (cell < 0) return;
  const unsigned int r = 0xffffffffu - (unsigned int)(a.repkey[cell] & 0xffffffffull);
  if ((long long)r == i) return;                                   // the representative itself
  float tu[3], tv[3];
  frame_uv(reinterpret_cast<const float4*>(a.quat)[r], tu, tv);
  const float d0 = __fsub_rn(a.mean[3 * i], a.mean[3 * r]), d1 = __fsub_rn(a.mean[3 * i + 1], a.mean[3 * r + 1]),
              d2 = __fsub_rn(a.mean[3 * i + 2], a.mean[3 * r + 2]);
  const float u = __fdiv_rn(__fadd_rn(__fadd_rn(__fmul_rn(tu[0], d0), __fmul_rn(tu[1], d1)), __fmul_rn(tu[2], d2)), a.scale[2 * r]);
  const float v = __fdiv_rn(__fadd_rn(__fadd_rn(__fmul_rn(tv[0], d0), __fmul_rn(tv[1], d1)), __fmul_rn(tv[2], d2)), a.scale[2 * r + 1]);
  const unsigned int bits = __float_as_uint(__fadd_rn(__fmul_rn(u, u), __fmul_rn(v, v)));
  const unsigned int pos = a.start[cell] + atomicAdd(&a.cursor[cell], 1u);
  a.keys0[pos] = bits; a.vals0[pos] = (unsigned int)i;
  a.rho2[i] = bits;
}

// per cell: the q_cover-quantile of the members' rho^2 (sorted segment), the cover radius, the representative's new scale
__global__ void __launch_bounds__(kMT) cover_cell_kernel(const CoverArgs a) {
  const long long g = (long long)blockIdx.x * kMT + threadIdx.x;
  if (g >= a.ncell) return;
  const unsigned int nc = a.cnt[g];
  if (nc < 2u) return;
  const int n = (int)nc - 1;
  int k = __float2int_ru(__fmul_rn(a.P.q_cover, (float)n));
  k = min(max(k, 1), n);
  const float Q = __uint_as_float(a.keys0[a.start[g] + (unsigned int)(k - 1)]);
  const float R2 = fmaxf(__fmul_rn(a.P.kappa, a.P.kappa), Q);
  a.R2[g] = R2;
  const float f = __fdiv_rn(__fsqrt_rn(R2), a.P.kappa);
  const unsigned int r = 0xffffffffu - (unsigned int)(a.repkey[g] & 0xffffffffull);
  const float n0 = fminf(__fmul_rn(f, a.scale[2 * r]), a.P.s_max), n1 = fminf(__fmul_rn(f, a.scale[2 * r + 1]), a.P.s_max);
  a.scale[2 * r] = n0; a.scale[2 * r + 1] = n1;
  if (a.log_scale) { a.log_scale[2 * r] = logf(n0); a.log_scale[2 * r + 1] = logf(n1); }
}

__device__ __forceinline__ bool cover_redundant(const CoverArgs& a, long long i) {
  if (i >= a.N) return false;
  const int cell = a.cellid[i];
  if (cell < 0 || a.cnt[cell] < 2u) return false;
  const unsigned int r = 0xffffffffu - (unsigned int)(a.repkey[cell] & 0xffffffffull);
  if ((long long)r == i) return false;
  return __uint_as_float(a.rho2[i]) <= a.R2[cell];
}

__global__ void __launch_bounds__(kMT) cover_count_kernel(const CoverArgs a) {
  const long long i = (long long)blockIdx.x * kMT + threadIdx.x;
  const unsigned int n = (unsigned int)__syncthreads_count(cover_redundant(a, i));
  if (threadIdx.x == 0) a.blk[blockIdx.x] = n;
}

__global__ void __launch_bounds__(kMT) cover_flag_kernel(const CoverArgs a) {
  __shared__ unsigned int s_w[kMT / 32];
  const long long i = (long long)blockIdx.x * kMT + threadIdx.x;
  const bool red = cover_redundant(a, i);
  const unsigned int rank = a.blk[blockIdx.x] + block_rank(red, s_w);
  if (i < a.N) a.keep[i] = (red && rank < a.P.cap) ? 0 : 1;          // the cap keeps the removals of lowest index (R36)
  if (blockIdx.x == 0 && threadIdx.x == 0) *a.n_removed = (long long)min(a.tot[0], a.P.cap);
}

struct CoverWs {
  int* cellid; unsigned int* rho2; unsigned long long* repkey; unsigned int* cnt; unsigned int* start; unsigned int* cursor;
  unsigned int* ranges; float* R2; unsigned int* keys0; unsigned int* keys1; unsigned int* vals0; unsigned int* vals1;
  unsigned int* blk; unsigned int* tot; size_t zero_begin, zero_end, total;
};
CoverWs carve_cover(char* p0, int64_t N, int64_t ncell) {
  const size_t Nn = (size_t)(N > 0 ? N : 1), C = (size_t)(ncell > 0 ? ncell : 1);
  const size_t nb = (Nn + kMT - 1) / kMT + 1;
  CoverWs w;
  size_t o = 0;
  auto take = [&](size_t bytes) { char* q = p0 ? p0 + o : nullptr; o += align_up(bytes); return q; };
  w.zero_begin = o;
  w.repkey = reinterpret_cast<unsigned long long*>(take(C * 8));
  w.cnt = reinterpret_cast<unsigned int*>(take(C * 4));
  w.cursor = reinterpret_cast<unsigned int*>(take(C * 4));
  w.zero_end = o;
  w.start = reinterpret_cast<unsigned int*>(take(C * 4));
  w.ranges = reinterpret_cast<unsigned int*>(take(C * 8));
  w.R2 = reinterpret_cast<float*>(take(C * 4));
  w.cellid = reinterpret_cast<int*>(take(Nn * 4));
  w.rho2 = reinterpret_cast<unsigned int*>(take(Nn * 4));
  w.keys0 = reinterpret_cast<unsigned int*>(take(Nn * 4));
  w.keys1 = reinterpret_cast<unsigned int*>(take(Nn * 4));
  w.vals0 = reinterpret_cast<unsigned int*>(take(Nn * 4));
  w.vals1 = reinterpret_cast<unsigned int*>(take(Nn * 4));
  w.blk = reinterpret_cast<unsigned int*>(take(nb * 4));
  w.tot = reinterpret_cast<unsigned int*>(take(256));
  w.total = o;
  return w;
}

}  // namespace

size_t cover_workspace_bytes(int64_t N, int64_t ncells) { return carve_cover(nullptr, N, ncells).total; }

cudaError_t launch_cover_prune(int64_t N, const float* mean, const float* quat, float* scale, float* log_scale,
                               const float* opacity, const float* c, const float* thr, const CoverParams& P,
                               unsigned char* keep, long long* n_removed, void* workspace, cudaStream_t st) {
  const long long ncell = (long long)P.dim_a * P.dim_b;
  const CoverWs w = carve_cover(static_cast<char*>(workspace), N, ncell);
  cudaError_t e = cudaMemsetAsync(static_cast<char*>(workspace) + w.zero_begin, 0, w.zero_end - w.zero_begin, st);
  if (e != cudaSuccess) return e;
  CoverArgs a;
  a.N = N; a.mean = mean; a.quat = quat; a.scale = scale; a.log_scale = log_scale; a.opacity = opacity; a.c = c; a.thr = thr;
  a.P = P; a.ncell = ncell; a.cellid = w.cellid; a.rho2 = w.rho2; a.repkey = w.repkey; a.cnt = w.cnt; a.start = w.start;
  a.cursor = w.cursor; a.ranges = w.ranges; a.R2 = w.R2; a.keys0 = w.keys0; a.vals0 = w.vals0; a.blk = w.blk; a.tot = w.tot;
  a.keep = keep; a.n_removed = n_removed;
  const unsigned gn = (unsigned)((N + kMT - 1) / kMT), gc = (unsigned)((ncell + kMT - 1) / kMT);
  if (gn) cover_assign_kernel<<<gn, kMT, 0, st>>>(a);
  cover_members_count_kernel<<<gc, kMT, 0, st>>>(a);
  scan_blocks_kernel<<<1, 1024, 0, st>>>(w.start, nullptr, ncell, w.tot + 1, nullptr);
  cover_ranges_kernel<<<gc, kMT, 0, st>>>(a);
  if (gn) cover_member_kernel<<<gn, kMT, 0, st>>>(a);
  e = launch_tile_sort(w.keys0, w.keys1, w.vals0, w.vals1, nullptr, w.ranges, nullptr, nullptr, (int)ncell, st);
  if (e != cudaSuccess) return e;
  cover_cell_kernel<<<gc, kMT, 0, st>>>(a);
  if (gn) cover_count_kernel<<<gn, kMT, 0, st>>>(a);
  scan_blocks_kernel<<<1, 1024, 0, st>>>(w.blk, nullptr, (long long)gn, w.tot, nullptr);
  cover_flag_kernel<<<gn ? gn : 1, kMT, 0, st>>>(a);
  return cudaGetLastError();
}

}  // namespace lgs
