// K3: hand-written segmented sort (step S3 of SURVEY.md 8(a), north_star (2): "tile-key emission
// (tile_id, range) plus a hand-written radix sort and tile-range build").
//
// The emission kernel buckets the keys by tile (the most significant digit of the (tile_id, range)
// key) directly into the tile's [start, end) segment, in arbitrary order -- that is the first radix
// step of the sort.  What is left is, per tile, a sort by the 32 range bits with ties broken by
// surfel index -- which is exactly the order a stable sort of the (tile_id << 32 | range bits) keys
// emitted in surfel-index order produces.  The tile lengths are
// heavy-tailed (config 2: median 117, mean 310, max 2,309), so two kernels share the tiles by length
// class, each one CTA per tile:
//   small class (n < kBigMin, 128 threads):
//     n <= kBitonicMax : bitonic network on the 64-bit composites (range bits << 32 | surfel id) in
//                        shared memory, every compare-exchange ascending (the first step of a merge
//                        mirrors its partner), so a list of any length runs the network of the next
//                        power of two minus the comparators that reach past n; steps with partner
//                        distance <= 32 stay inside one warp's 64 elements and need no block barrier.
//     else             : LSD radix sort in shared memory, items held in registers between passes.
//   big class (n >= kBigMin, 512 threads): the same radix sort with wider digits; lists longer than
//     kBigSmem ping-pong between the two global buffers (8-bit digits, per-chunk ranking).
// The radix sort looks at the bits that actually vary over the list (OR of key ^ key[0]) and splits
// that span evenly over as few passes as the class's digit width allows -- the exponent byte of a
// tile's ranges is almost constant.  A pass ranks with warp match-any, takes the digit totals from
// the per-warp counts (no separate histogram), and scatters in place (every thread holds its items
// in registers).  The radix paths end with a pass that orders runs of equal range bits by surfel
// index (the input order inside a segment is arbitrary).  Measured alternatives (B200, config 2):
// one 256-thread radix kernel for all tiles 46 us; bitonic network for every list <= 4096: 57 us
// (log^2 n stages of ~20 instructions per comparator cost more than 3-4 radix passes beyond ~256
// keys); this split: 42 us, bound by the latency of the longest lists of each class.
#include "lgs_internal.cuh"

namespace lgs {
namespace {

constexpr int kBitonicMax = 256;
constexpr int kSmallThreads = 128, kSmallBits = 7;       // n <  kBigMin: 128 bins, one digit per thread
constexpr int kBigThreads = 512, kBigBits = 9;           // n >= kBigMin: 512 bins, one digit per thread
constexpr int kBigMin = 1 << (kSortBigBucket - 1);        // 1024: first length of the big class
constexpr int kBigSmem = 4096;                           // longest list sorted in shared memory
constexpr int kItems = 8;                                // items per thread (both classes)
static_assert(kSmallThreads * kItems >= kBigMin - 1 && kBigThreads * kItems >= kBigSmem, "class capacities");

struct TieShared { unsigned int first, end; };      // order_ties: the long run being sorted

template <int THREADS, int BITS>
struct SortShared {
  unsigned int wh[THREADS / 32][1 << BITS];   // per-warp digit counts -> scatter offsets
  unsigned int tb[THREADS];                   // exclusive base of each thread's digit group
  unsigned int wsum[THREADS / 32];
  TieShared tie;
};

__device__ __forceinline__ void cmpxchg(unsigned long long* e, int i, int l) {
  const unsigned long long x = e[i], y = e[l];
  if (x > y) { e[i] = y; e[l] = x; }
}

// Sorts (keys, vals)[0, n) by (key, val); e = shared array of >= n 64-bit words.  Comparator t of a stage is
// handled by thread t % THREADS in every stage, so a warp keeps touching the same 64-element windows as long as the partner distance stays <= 32.
// kv != NULL: the unsorted input is read from the interleaved (key, value) pairs kv[0, n) instead of (keys, vals).
template <int THREADS>
__device__ __forceinline__ void bitonic_sort(unsigned int* keys, unsigned int* vals, const uint2* kv, int n,
                                             unsigned long long* e, int tid) {
  int P = 64;
  while (P < n) P <<= 1;
  if (kv) {
    for (int i = tid; i < n; i += THREADS) { const uint2 t = kv[i]; e[i] = ((unsigned long long)t.x << 32) | t.y; }
  } else {
    for (int i = tid; i < n; i += THREADS) e[i] = ((unsigned long long)keys[i] << 32) | vals[i];
  }
  const int half = P >> 1;
  bool prev_cross = true;                      // the fill above was strided over the whole block
  for (int k = 2; k <= P; k <<= 1) {
    {                                          // merge step 1: partner mirrored inside the block of k
      const int j = k >> 1;
      const bool cross = j > 32;
      if (cross || prev_cross) __syncthreads(); else __syncwarp();
      prev_cross = cross;
      for (int t = tid; t < half; t += THREADS) {
        const int off = t & (j - 1);
        const int i = ((t - off) << 1) + off;
        const int l = ((t - off) << 1) + (k - 1 - off);
        if (l < n) cmpxchg(e, i, l);
      }
    }
    for (int j = k >> 2; j >= 1; j >>= 1) {    // remaining steps: partner at distance j
      const bool cross = j > 32;
      if (cross || prev_cross) __syncthreads(); else __syncwarp();
      prev_cross = cross;
      for (int t = tid; t < half; t += THREADS) {
        const int i = ((t & ~(j - 1)) << 1) | (t & (j - 1));
        const int l = i | j;
        if (l < n) cmpxchg(e, i, l);
      }
    }
  }
  __syncthreads();
  for (int i = tid; i < n; i += THREADS) {
    const unsigned long long v = e[i];
    keys[i] = (unsigned int)(v >> 32);
    vals[i] = (unsigned int)v;
  }
}

// Orders runs of equal range bits by surfel index.  Short runs (the normal case: a handful of surfels at one fp32
// range) are insertion-sorted by the thread that owns the run's head; runs longer than kTieSerial -- a map with many
// surfels at one range in one tile, e.g. a sphere shell or a quantised map -- are listed and then sorted by the whole
// CTA with the all-ascending bitonic network (O(L log^2 L / threads) instead of O(L^2) in one thread).  All threads of
// the CTA must call it (block barriers inside).
constexpr int kTieSerial = 16;
__device__ __forceinline__ void bitonic_values(unsigned int* v, int n, int tid, int nthreads) {
  int P = 2;
  while (P < n) P <<= 1;
  const int half = P >> 1;
  for (int k = 2; k <= P; k <<= 1) {
    __syncthreads();
    for (int t = tid; t < half; t += nthreads) {     // merge step 1: partner mirrored inside the block of k
      const int j = k >> 1, off = t & (j - 1);
      const int i = ((t - off) << 1) + off, l = ((t - off) << 1) + (k - 1 - off);
      if (l < n) { const unsigned int x = v[i], y = v[l]; if (x > y) { v[i] = y; v[l] = x; } }
    }
    for (int j = k >> 2; j >= 1; j >>= 1) {          // remaining steps: partner at distance j
      __syncthreads();
      for (int t = tid; t < half; t += nthreads) {
        const int i = ((t & ~(j - 1)) << 1) | (t & (j - 1)), l = i | j;
        if (l < n) { const unsigned int x = v[i], y = v[l]; if (x > y) { v[i] = y; v[l] = x; } }
      }
    }
  }
  __syncthreads();
}

__device__ __forceinline__ void order_ties(const unsigned int* sk, unsigned int* sv, int n, int tid, int nthreads,
                                           TieShared& T) {
  unsigned int pos = 0;                // long runs that start before pos are sorted (uniform over the CTA)
  for (bool first_sweep = true;; first_sweep = false) {
    if (tid == 0) { T.first = 0xffffffffu; T.end = 0u; }
    __syncthreads();
    for (int i = tid; i + 1 < n; i += nthreads) {
      const unsigned int k = sk[i];
      if (sk[i + 1] == k && (i == 0 || sk[i - 1] != k)) {          // head of a run
        if (i + kTieSerial < n && sk[i + kTieSerial] == k) {       // (sorted keys: the run is longer than kTieSerial)
          if ((unsigned int)i >= pos) atomicMin(&T.first, (unsigned int)i);
        } else if (first_sweep) {
          int e = i + 2;
          while (e < n && sk[e] == k) ++e;
          for (int p = i + 1; p < e; ++p) {
            const unsigned int v = sv[p];
            int q = p - 1;
            while (q >= i && sv[q] > v) { sv[q + 1] = sv[q]; --q; }
            sv[q + 1] = v;
          }
        }
      }
    }
    __syncthreads();
    const unsigned int lo = T.first;
    if (lo == 0xffffffffu) break;                                   // (the normal case: no long run, one sweep)
    {
      const unsigned int k = sk[lo];
      unsigned int e = 0u;
      for (int j = (int)lo + tid; j < n; j += nthreads) if (sk[j] == k) e = (unsigned int)j + 1u;
      if (e) atomicMax(&T.end, e);
    }
    __syncthreads();
    const unsigned int hi = T.end;
    bitonic_values(sv + lo, (int)(hi - lo), tid, nthreads);
    pos = hi;
  }
}

// ---- radix sort of one list in shared memory; n <= THREADS * kItems ------------------------------
template <int THREADS, int BITS>
__device__ __forceinline__ void radix_smem(unsigned int* keys, unsigned int* vals, const uint2* kv, int n,
                                           unsigned int* ek, unsigned int* ev, SortShared<THREADS, BITS>& S, int tid) {
  constexpr int NW = THREADS / 32;
  constexpr int kThreadsLog = (THREADS == 512) ? 9 : (THREADS == 256) ? 8 : 7;
  static_assert((1 << kThreadsLog) == THREADS, "THREADS must be 128, 256 or 512");
  const int lane = tid & 31, warp = tid >> 5;
  // items per thread for THIS list (1..kItems): the list is spread evenly over the warps, so that the
  // sequential part of a pass (ranking item after item) is as short as the list allows
  const int ipt = (n + THREADS - 1) / THREADS;
  const int wbase = warp * (32 * ipt);
  unsigned int key[kItems], val[kItems];
  const unsigned int key0 = kv ? kv[0].x : keys[0];
  unsigned int v = 0;
#pragma unroll
  for (int j = 0; j < kItems; ++j) {
    if (j >= ipt) break;
    const int idx = wbase + j * 32 + lane;
    const bool valid = idx < n;
    key[j] = 0xffffffffu; val[j] = 0xffffffffu;
    if (valid) {
      if (kv) { const uint2 t = kv[idx]; key[j] = t.x; val[j] = t.y; }
      else { key[j] = keys[idx]; val[j] = vals[idx]; }
    }
    v |= valid ? (key[j] ^ key0) : 0u;
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v |= __shfl_xor_sync(0xffffffffu, v, o);
  if (lane == 0) S.wsum[warp] = v;
  __syncthreads();
  unsigned int vary = 0;
#pragma unroll
  for (int w = 0; w < NW; ++w) vary |= S.wsum[w];
  // bits [lo, hi) vary; npass digits of b bits each cover them
  const int hi = 32 - __clz(vary), lo = vary ? (__ffs(vary) - 1) : 0;
  const int span = hi - lo;
  const int npass = (span + BITS - 1) / BITS;
  const int b = npass ? (span + npass - 1) / npass : 0;
  const unsigned int nb = 1u << b, dmask = nb - 1u;
  // digit ownership in the offsets phase: thread t owns digits [t * nbpt, (t + 1) * nbpt)
  const int nbpt_log = b > kThreadsLog ? b - kThreadsLog : 0;
  const int nbpt = 1 << nbpt_log;
  const int nact = (int)nb >> nbpt_log;
  if (npass == 0) {                          // every key equal: only the tie pass has work
#pragma unroll
    for (int j = 0; j < kItems; ++j) {
      if (j >= ipt) break;
      const int idx = wbase + j * 32 + lane;
      if (idx < n) { ek[idx] = key[j]; ev[idx] = val[j]; }
    }
  }
  for (int pass = 0; pass < npass; ++pass) {
    const int shift = lo + pass * b;
    for (unsigned int d = lane; d < nb; d += 32) S.wh[warp][d] = 0;     // own row only
    __syncwarp();
    // ---- per-warp ranking (memory order == warp, item, lane): pk = digit | rank << 16 ---------
    unsigned int pk[kItems];
#pragma unroll
    for (int j = 0; j < kItems; ++j) {
      if (j >= ipt) break;
      const bool valid = wbase + j * 32 + lane < n;
      const unsigned int d = valid ? ((key[j] >> shift) & dmask) : 0xffffu;
      const unsigned int peers = __match_any_sync(0xffffffffu, d);
      const unsigned int below = __popc(peers & ((1u << lane) - 1u));
      unsigned int pre = 0;
      if (valid && below == 0) pre = atomicAdd(&S.wh[warp][d], (unsigned int)__popc(peers));
      __syncwarp();
      pre = __shfl_sync(0xffffffffu, pre, __ffs(peers) - 1);
      pk[j] = d | ((pre + below) << 16);
    }
    __syncthreads();
    // ---- offsets: wh[w][d] <- (digits before d in the owner's group) + (warps before w); tb <- group base
    unsigned int local = 0;
    if (tid < nact) {
      for (int i = 0; i < nbpt; ++i) {
        const int d = tid * nbpt + i;
        unsigned int t = 0;
#pragma unroll
        for (int w = 0; w < NW; ++w) {
          const unsigned int c = S.wh[w][d];
          S.wh[w][d] = local + t;
          t += c;
        }
        local += t;
      }
    }
    unsigned int inc = local;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const unsigned int u = __shfl_up_sync(0xffffffffu, inc, o);
      if (lane >= o) inc += u;
    }
    if (lane == 31) S.wsum[warp] = inc;
    __syncthreads();
    unsigned int woff = 0;
#pragma unroll
    for (int w = 0; w < NW; ++w) woff += (w < warp) ? S.wsum[w] : 0u;
    S.tb[tid] = woff + inc - local;
    __syncthreads();
    // ---- scatter in place (every item is in a register), then pick the items up in the new order
#pragma unroll
    for (int j = 0; j < kItems; ++j) {
      if (j >= ipt) break;
      const unsigned int d = pk[j] & 0xffffu;
      if (d != 0xffffu) {
        const unsigned int pos = S.wh[warp][d] + S.tb[d >> nbpt_log] + (pk[j] >> 16);
        ek[pos] = key[j];
        ev[pos] = val[j];
      }
    }
    __syncthreads();
    if (pass + 1 < npass) {
#pragma unroll
      for (int j = 0; j < kItems; ++j) {
        if (j >= ipt) break;
        const int idx = wbase + j * 32 + lane;
        if (idx < n) { key[j] = ek[idx]; val[j] = ev[idx]; }
      }
    }
  }
  if (npass == 0) __syncthreads();
  order_ties(ek, ev, n, tid, THREADS, S.tie);
  __syncthreads();
  for (int i = tid; i < n; i += THREADS) { keys[i] = ek[i]; vals[i] = ev[i]; }
}

// ---- lists longer than kBigSmem: stable 8-bit LSD passes between the two global buffers ----------
struct GlobalShared {
  unsigned int wh[kBigThreads / 32][256];
  unsigned int hist[256];
  unsigned int cbase[256];
  unsigned int scan[8];
  unsigned int vary;
  TieShared tie;
};

__device__ __forceinline__ void radix_pass_global(const unsigned int* sk, const unsigned int* sv, unsigned int* dk,
                                                  unsigned int* dv, int n, int shift, GlobalShared& S, int tid) {
  constexpr int NW = kBigThreads / 32, kChunk = kBigThreads * kItems;
  const int lane = tid & 31, warp = tid >> 5;
  if (tid < 256) S.hist[tid] = 0;
  __syncthreads();
  for (int i = tid; i < n; i += kBigThreads) atomicAdd(&S.hist[(sk[i] >> shift) & 255u], 1u);
  __syncthreads();
  const unsigned int h = (tid < 256) ? S.hist[tid] : 0u;
  unsigned int inc = h;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const unsigned int v = __shfl_up_sync(0xffffffffu, inc, o);
    if (lane >= o) inc += v;
  }
  if (lane == 31 && warp < 8) S.scan[warp] = inc;
  __syncthreads();
  unsigned int woff = 0;
#pragma unroll
  for (int w = 0; w < 8; ++w) woff += (w < warp) ? S.scan[w] : 0u;
  if (tid < 256) S.hist[tid] = woff + inc - h;  // running base of digit `tid`
  for (int c0 = 0; c0 < n; c0 += kChunk) {
    const int nc = min(kChunk, n - c0);
    for (int k = tid; k < NW * 256; k += kBigThreads) (&S.wh[0][0])[k] = 0;
    __syncthreads();
    const int wbase = c0 + warp * (32 * kItems);
    unsigned int key[kItems], rank[kItems], dig[kItems];
#pragma unroll
    for (int j = 0; j < kItems; ++j) {
      const int idx = wbase + j * 32 + lane;
      const bool valid = idx < c0 + nc;
      key[j] = valid ? sk[idx] : 0u;
      dig[j] = valid ? ((key[j] >> shift) & 255u) : 256u;
    }
#pragma unroll
    for (int j = 0; j < kItems; ++j) {
      const unsigned int d = dig[j];
      const unsigned int peers = __match_any_sync(0xffffffffu, d);
      const unsigned int below = __popc(peers & ((1u << lane) - 1u));
      unsigned int pre = 0;
      if (d < 256u && below == 0) pre = atomicAdd(&S.wh[warp][d], (unsigned int)__popc(peers));
      __syncwarp();
      rank[j] = __shfl_sync(0xffffffffu, pre, __ffs(peers) - 1) + below;
    }
    __syncthreads();
    if (tid < 256) {
      unsigned int cnt = 0;
#pragma unroll
      for (int w = 0; w < NW; ++w) {
        const unsigned int c = S.wh[w][tid];
        S.wh[w][tid] = cnt;
        cnt += c;
      }
      const unsigned int b = S.hist[tid];
      S.cbase[tid] = b;
      S.hist[tid] = b + cnt;
    }
    __syncthreads();
#pragma unroll
    for (int j = 0; j < kItems; ++j) {
      const unsigned int d = dig[j];
      if (d < 256u) {
        const unsigned int pos = S.cbase[d] + S.wh[warp][d] + rank[j];
        dk[pos] = key[j];
        dv[pos] = sv[wbase + j * 32 + lane];
      }
    }
    __syncthreads();
  }
}

__device__ __forceinline__ void radix_global(unsigned int* keys, unsigned int* vals, const uint2* kv, unsigned int* tk,
                                             unsigned int* tv, int n, GlobalShared& S, int tid) {
  if (kv) {                                   // split the interleaved input first (lists > kBigSmem keys are rare)
    for (int i = tid; i < n; i += kBigThreads) { const uint2 t = kv[i]; keys[i] = t.x; vals[i] = t.y; }
    __syncthreads();
  }
  unsigned int *sk = keys, *sv = vals, *dk = tk, *dv = tv;
  if (tid == 0) S.vary = 0u;
  __syncthreads();
  {
    const unsigned int k0 = sk[0];
    unsigned int v = 0;
    for (int i = tid; i < n; i += kBigThreads) v |= sk[i] ^ k0;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v |= __shfl_xor_sync(0xffffffffu, v, o);
    if ((tid & 31) == 0 && v) atomicOr(&S.vary, v);
  }
  __syncthreads();
  const unsigned int vary = S.vary;
  for (int pass = 0; pass < 4; ++pass) {
    const int shift = pass * 8;
    if (((vary >> shift) & 255u) == 0u) continue;     // the digit is the same in every key
    radix_pass_global(sk, sv, dk, dv, n, shift, S, tid);
    unsigned int* t;
    t = sk; sk = dk; dk = t;
    t = sv; sv = dv; dv = t;
  }
  __syncthreads();
  order_ties(sk, sv, n, tid, kBigThreads, S.tie);
  if (sk != keys) {
    __syncthreads();
    for (int i = tid; i < n; i += kBigThreads) { keys[i] = sk[i]; vals[i] = sv[i]; }
  }
}

// ---- kernels -------------------------------------------------------------------------------------
// Small class: one CTA per segment of the schedule; segments of the big class are skipped.
__global__ void __launch_bounds__(kSmallThreads) tile_sort_small_kernel(unsigned int* keys0, unsigned int* vals0,
                                                                        const uint2* kv,
                                                                        const unsigned int* __restrict__ ranges,
                                                                        const uint4* __restrict__ sched) {
  __shared__ __align__(16) unsigned int s_list[2 * kSmallThreads * kItems];
  __shared__ SortShared<kSmallThreads, kSmallBits> S;
  const int tid = threadIdx.x;
  unsigned int start;
  int n;
  if (sched) { const uint4 e = sched[blockIdx.x]; start = e.y; n = (int)(e.z - e.y); }
  else { start = ranges[2 * blockIdx.x]; n = (int)(ranges[2 * blockIdx.x + 1] - start); }
  const uint2* kvs = kv ? kv + start : nullptr;
  if (n > 1 && n < kBigMin) {
    if (n <= kBitonicMax)
      bitonic_sort<kSmallThreads>(keys0 + start, vals0 + start, kvs, n, reinterpret_cast<unsigned long long*>(s_list), tid);
    else
      radix_smem<kSmallThreads, kSmallBits>(keys0 + start, vals0 + start, kvs, n, s_list, s_list + kSmallThreads * kItems, S, tid);
  } else if (n == 1 && kv) {
    if (tid == 0) { const uint2 t = kvs[0]; keys0[start] = t.x; vals0[start] = t.y; }
  }
  // This grid is launched with programmatic stream serialisation while the big-class grid is still
  // running (the two sort disjoint segments).  No CTA may retire before the big-class grid has
  // completed, or the next kernel in the stream could start on unsorted long lists.
  asm volatile("griddepcontrol.wait;" ::: "memory");
}

// Big class: the schedule lists the segments longest first, so the big ones are its first *n_big
// entries (n_big == NULL: look at every segment); CTAs stride over them.
__global__ void __launch_bounds__(kBigThreads) tile_sort_big_kernel(unsigned int* keys0, unsigned int* keys1,
                                                                    unsigned int* vals0, unsigned int* vals1,
                                                                    const uint2* kv,
                                                                    const unsigned int* __restrict__ ranges,
                                                                    const uint4* __restrict__ sched, int nseg,
                                                                    const unsigned int* __restrict__ n_big) {
  extern __shared__ __align__(16) unsigned int s_dyn[];      // list (2 x kBigSmem words), then SortShared
  unsigned int* s_list = s_dyn;
  SortShared<kBigThreads, kBigBits>& S = *reinterpret_cast<SortShared<kBigThreads, kBigBits>*>(s_dyn + 2 * kBigSmem);
  static_assert(sizeof(GlobalShared) <= sizeof(unsigned int) * 2 * kBigSmem, "GlobalShared aliases the list buffer");
  const int tid = threadIdx.x;
  asm volatile("griddepcontrol.launch_dependents;");    // the small-class grid may start right away
  const int limit = n_big ? min((int)*n_big, nseg) : nseg;
  for (int b = blockIdx.x; b < limit; b += gridDim.x) {
    unsigned int start;
    int n;
    if (sched) { const uint4 e = sched[b]; start = e.y; n = (int)(e.z - e.y); }
    else { start = ranges[2 * b]; n = (int)(ranges[2 * b + 1] - start); }
    if (n < kBigMin) continue;
    __syncthreads();                                   // the previous segment's reads of shared memory are done
    const uint2* kvs = kv ? kv + start : nullptr;
    if (n <= kBigSmem) radix_smem<kBigThreads, kBigBits>(keys0 + start, vals0 + start, kvs, n, s_list, s_list + kBigSmem, S, tid);
    else radix_global(keys0 + start, vals0 + start, kvs, keys1 + start, vals1 + start, n, *reinterpret_cast<GlobalShared*>(s_list), tid);
  }
}

}  // namespace

cudaError_t launch_tile_sort(uint32_t* keys0, uint32_t* keys1, uint32_t* vals0, uint32_t* vals1, const uint2* kv,
                             const unsigned int* ranges, const uint4* sched, const unsigned int* n_big, int nseg,
                             cudaStream_t st) {
  if (nseg <= 0) return cudaSuccess;
  const size_t dyn = sizeof(unsigned int) * 2 * kBigSmem + sizeof(SortShared<kBigThreads, kBigBits>);
  // (the attribute is per device: set it on every call -- it is a cheap host-side call -- instead of caching a flag
  // that would be wrong for the second device of a process)
  cudaError_t e = cudaFuncSetAttribute(tile_sort_big_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dyn);
  if (e != cudaSuccess) return e;
  const int big_grid = min(nseg, sm_count() * 3);
  tile_sort_big_kernel<<<big_grid, kBigThreads, dyn, st>>>(keys0, keys1, vals0, vals1, kv, ranges, sched, nseg, n_big);
  const unsigned int* r = ranges; const uint4* o = sched;
  e = launch_pdl(tile_sort_small_kernel, dim3((unsigned)nseg), dim3(kSmallThreads), 0, st, keys0, vals0, kv, r, o);
  if (e != cudaSuccess) return e;
  return cudaGetLastError();
}

}  // namespace lgs
