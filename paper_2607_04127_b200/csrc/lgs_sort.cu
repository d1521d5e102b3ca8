// K3: hand-written stable LSD radix sort of (key64, val32) pairs (step S3 of SURVEY.md 8(a),
// north_star (2): "tile-key emission (tile_id, range) plus a hand-written radix sort").
//
// One histogram kernel for all digits, then one single-pass kernel per 8-bit digit:
// every CTA ranks its 2048 keys with warp match-any multisplit, obtains its global
// per-digit base by decoupled look-back over the preceding CTAs' counts (ticket order),
// and scatters.  The number of keys lives on the device (no host sync); grids are sized
// for the capacity and surplus CTAs exit.
#include "lgs_internal.cuh"

namespace lgs {
namespace {

constexpr unsigned int kAgg = 1u << 30, kPre = 2u << 30, kCntMask = (1u << 30) - 1u;

__global__ void __launch_bounds__(kSortThreads) sort_hist_kernel(const unsigned long long* __restrict__ keys,
                                                                 const unsigned int* __restrict__ n_dev, int passes,
                                                                 unsigned int* __restrict__ hist) {
  __shared__ unsigned int sh[kMaxPasses * kRadix];
  const unsigned int n = *n_dev;
  const long long base = (long long)blockIdx.x * kSortTile;
  if (base >= (long long)n) return;
  for (int t = threadIdx.x; t < passes * kRadix; t += kSortThreads) sh[t] = 0;
  __syncthreads();
#pragma unroll
  for (int j = 0; j < kSortItems; ++j) {
    const long long idx = base + j * kSortThreads + threadIdx.x;
    if (idx < (long long)n) {
      const unsigned long long k = keys[idx];
      for (int p = 0; p < passes; ++p) atomicAdd(&sh[p * kRadix + (unsigned int)((k >> (p * kRadixBits)) & (kRadix - 1))], 1u);
    }
  }
  __syncthreads();
  for (int t = threadIdx.x; t < passes * kRadix; t += kSortThreads) {
    const unsigned int c = sh[t];
    if (c) atomicAdd(&hist[t], c);
  }
}

__global__ void __launch_bounds__(kSortThreads) sort_pass_kernel(const unsigned long long* __restrict__ kin,
                                                                 const unsigned int* __restrict__ vin,
                                                                 unsigned long long* __restrict__ kout,
                                                                 unsigned int* __restrict__ vout,
                                                                 const unsigned int* __restrict__ n_dev, int pass,
                                                                 const unsigned int* __restrict__ hist,
                                                                 unsigned int* status, unsigned int* ticket) {
  __shared__ unsigned int s_wh[kSortThreads / 32][kRadix];   // per-warp digit counts -> exclusive offsets
  __shared__ unsigned int s_base[kRadix];                    // global base of this CTA's run of each digit
  __shared__ unsigned int s_scan[kSortThreads / 32];
  __shared__ unsigned int s_tile;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const unsigned int n = *n_dev;
  const unsigned int n_tiles = (n + kSortTile - 1) / kSortTile;
  if (tid == 0) s_tile = atomicAdd(ticket, 1u);
#pragma unroll
  for (int w = 0; w < kSortThreads / 32; ++w) s_wh[w][tid] = 0;
  __syncthreads();
  const unsigned int tile = s_tile;
  if (tile >= n_tiles) return;
  const int shift = pass * kRadixBits;

  // ---- load + per-warp ranking (memory order == warp, item, lane) -----------------------
  const long long wbase = (long long)tile * kSortTile + (long long)warp * (32 * kSortItems);
  unsigned long long key[kSortItems];
  unsigned int rank[kSortItems];
  unsigned int dig[kSortItems];
#pragma unroll
  for (int j = 0; j < kSortItems; ++j) {
    const long long idx = wbase + j * 32 + lane;
    const bool valid = idx < (long long)n;
    key[j] = valid ? kin[idx] : 0ull;
    dig[j] = valid ? (unsigned int)((key[j] >> shift) & (kRadix - 1)) : (unsigned int)kRadix;
  }
#pragma unroll
  for (int j = 0; j < kSortItems; ++j) {
    const unsigned int d = dig[j];
    const unsigned int peers = __match_any_sync(0xffffffffu, d);
    const unsigned int below = __popc(peers & ((1u << lane) - 1u));
    unsigned int pre = 0;
    if (d < (unsigned int)kRadix) pre = s_wh[warp][d];
    __syncwarp();
    if (d < (unsigned int)kRadix && below == 0) s_wh[warp][d] = pre + __popc(peers);
    __syncwarp();
    rank[j] = pre + below;
  }
  __syncthreads();

  // ---- per digit (thread d): exclusive offsets across warps, CTA count ---------------------
  unsigned int cnt = 0;
#pragma unroll
  for (int w = 0; w < kSortThreads / 32; ++w) {
    const unsigned int c = s_wh[w][tid];
    s_wh[w][tid] = cnt;
    cnt += c;
  }
  // ---- global start of digit d: exclusive scan of the digit histogram ----------------------
  const unsigned int h = hist[pass * kRadix + tid];
  unsigned int inc = h;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const unsigned int v = __shfl_up_sync(0xffffffffu, inc, o);
    if (lane >= o) inc += v;
  }
  if (lane == 31) s_scan[warp] = inc;
  // ---- publish this CTA's count, look back over the preceding tiles -------------------------
  unsigned int* my = status + (size_t)tile * kRadix + tid;
  *reinterpret_cast<volatile unsigned int*>(my) = (tile == 0 ? kPre : kAgg) | cnt;
  __syncthreads();
  unsigned int woff = 0;
  for (int w = 0; w < warp; ++w) woff += s_scan[w];
  const unsigned int digit_start = woff + inc - h;
  unsigned int excl = 0;
  if (tile > 0) {
    long long look = (long long)tile - 1;
    while (true) {
      const unsigned int v = *reinterpret_cast<volatile unsigned int*>(status + (size_t)look * kRadix + tid);
      const unsigned int flag = v >> 30;
      if (flag == 0u) continue;
      excl += v & kCntMask;
      if (flag == 2u) break;
      --look;
    }
    *reinterpret_cast<volatile unsigned int*>(my) = kPre | (excl + cnt);
  }
  s_base[tid] = digit_start + excl;
  __syncthreads();

  // ---- scatter ------------------------------------------------------------------------------
#pragma unroll
  for (int j = 0; j < kSortItems; ++j) {
    const unsigned int d = dig[j];
    if (d < (unsigned int)kRadix) {
      const unsigned int pos = s_base[d] + s_wh[warp][d] + rank[j];
      kout[pos] = key[j];
      vout[pos] = vin[wbase + j * 32 + lane];
    }
  }
}

}  // namespace

size_t sort_status_bytes(int64_t n, int passes) {
  const int64_t tiles = (n + kSortTile - 1) / kSortTile + 1;
  return (size_t)passes * (size_t)tiles * kRadix * sizeof(unsigned int);
}

// keys0/vals0 hold the input; result ends in buffer (passes & 1).  `hist` (passes*256),
// `status` (sort_status_bytes) and `tickets` (passes) must be zero on entry.
cudaError_t launch_sort(uint64_t* keys0, uint64_t* keys1, uint32_t* vals0, uint32_t* vals1, const unsigned int* n_dev,
                        int64_t n_max, int passes, unsigned int* hist, unsigned int* status, unsigned int* tickets,
                        cudaStream_t st) {
  if (n_max <= 0 || passes <= 0) return cudaSuccess;
  const unsigned int grid = (unsigned int)((n_max + kSortTile - 1) / kSortTile);
  const size_t tiles_stride = (size_t)(grid + 1) * kRadix;
  {
    ProfScope ps(LGS_PROF_SORT_HIST, st);
    sort_hist_kernel<<<grid, kSortThreads, 0, st>>>(reinterpret_cast<const unsigned long long*>(keys0), n_dev, passes, hist);
  }
  ProfScope ps(LGS_PROF_SORT_PASSES, st);
  unsigned long long* kb[2] = {reinterpret_cast<unsigned long long*>(keys0), reinterpret_cast<unsigned long long*>(keys1)};
  unsigned int* vb[2] = {vals0, vals1};
  for (int p = 0; p < passes; ++p) {
    sort_pass_kernel<<<grid, kSortThreads, 0, st>>>(kb[p & 1], vb[p & 1], kb[(p + 1) & 1], vb[(p + 1) & 1], n_dev, p,
                                                    hist, status + (size_t)p * tiles_stride, tickets + p);
  }
  return cudaGetLastError();
}

}  // namespace lgs
