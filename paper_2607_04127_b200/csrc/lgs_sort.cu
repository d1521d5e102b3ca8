// K3: hand-written segmented radix sort (step S3 of SURVEY.md 8(a), north_star (2): "tile-key
// emission (tile_id, range) plus a hand-written radix sort and tile-range build").
//
// The emission kernel buckets the keys by tile (the most significant digit of the (tile_id, range)
// key) directly into the tile's [start, end) segment, in arbitrary order.  What is left is, per
// tile, a sort by the 32 range bits with ties broken by surfel index -- which is exactly the order a
// stable sort of the (tile_id << 32 | range bits) keys emitted in surfel-index order produces
// (DESIGN.md "tile-list rule").  One CTA per tile: a stable LSD radix sort, four 8-bit digits, warp
// match-any ranking; lists up to kSortSmemCap entries never leave shared memory, longer ones
// ping-pong between the two global buffers (same code, generic pointers).  A final pass orders
// runs of equal range bits by surfel index (the input order inside a segment is arbitrary).
#include "lgs_internal.cuh"

namespace lgs {
namespace {

constexpr int kSortWarps = kSortThreads / 32;

__global__ void __launch_bounds__(kSortThreads) tile_sort_kernel(unsigned int* keys0, unsigned int* keys1,
                                                                 unsigned int* vals0, unsigned int* vals1,
                                                                 const unsigned int* __restrict__ ranges,
                                                                 const unsigned int* __restrict__ order) {
  extern __shared__ unsigned int s_buf[];                    // 4 x kSortSmemCap: keys A, vals A, keys B, vals B
  __shared__ unsigned int s_wh[kSortWarps][kRadix];          // per-warp digit counts -> exclusive offsets
  __shared__ unsigned int s_hist[kRadix];                    // digit histogram -> running global base
  __shared__ unsigned int s_cbase[kRadix];                   // base of the current super-chunk per digit
  __shared__ unsigned int s_scan[kRadix / 32];
  __shared__ unsigned int s_skip;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const unsigned int seg = order ? order[blockIdx.x] : blockIdx.x;
  const unsigned int start = ranges[2 * seg];
  const int n = (int)(ranges[2 * seg + 1] - start);
  if (n <= 1) return;
  const bool in_smem = n <= kSortSmemCap;
  unsigned int *sk, *sv, *dk, *dv;      // generic pointers: shared or global
  if (in_smem) {
    sk = s_buf; sv = s_buf + kSortSmemCap; dk = s_buf + 2 * kSortSmemCap; dv = s_buf + 3 * kSortSmemCap;
    for (int i = tid; i < n; i += kSortThreads) { sk[i] = keys0[start + i]; sv[i] = vals0[start + i]; }
  } else {
    sk = keys0 + start; sv = vals0 + start; dk = keys1 + start; dv = vals1 + start;
  }
  __syncthreads();

  for (int pass = 0; pass < 4; ++pass) {
    const int shift = pass * kRadixBits;
    if (tid < kRadix) s_hist[tid] = 0;
    if (tid == 0) s_skip = 0u;
    __syncthreads();
    for (int i = tid; i < n; i += kSortThreads) atomicAdd(&s_hist[(sk[i] >> shift) & (kRadix - 1)], 1u);
    __syncthreads();
    // a digit shared by every key of the segment (typical of the exponent byte) needs no pass
    if (tid < kRadix && s_hist[tid] == (unsigned int)n) s_skip = 1u;
    __syncthreads();
    if (s_skip) continue;
    // exclusive scan of the 256 digit counts (threads 0..255)
    unsigned int h = 0, inc = 0;
    if (tid < kRadix) {
      h = s_hist[tid];
      inc = h;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const unsigned int v = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += v;
      }
      if (lane == 31) s_scan[warp] = inc;
    }
    __syncthreads();
    if (tid < kRadix) {
      unsigned int woff = 0;
      for (int w = 0; w < warp; ++w) woff += s_scan[w];
      s_hist[tid] = woff + inc - h;                 // running base of digit `tid`
    }
    __syncthreads();

    for (int c0 = 0; c0 < n; c0 += kSortChunk) {
      const int nc = min(kSortChunk, n - c0);
      const int ipt = (nc + kSortThreads - 1) / kSortThreads;      // items per thread in this super-chunk
#pragma unroll
      for (int k = 0; k < kSortWarps * kRadix / kSortThreads; ++k) (&s_wh[0][0])[k * kSortThreads + tid] = 0;
      __syncthreads();
      // ---- load + per-warp ranking (memory order == warp, item, lane) -------------------------
      const int wbase = c0 + warp * (32 * ipt);
      unsigned int key[kSortItems], rank[kSortItems], dig[kSortItems];
#pragma unroll
      for (int j = 0; j < kSortItems; ++j) {
        const int idx = wbase + j * 32 + lane;
        const bool valid = j < ipt && idx < c0 + nc;
        key[j] = valid ? sk[idx] : 0u;
        dig[j] = valid ? ((key[j] >> shift) & (kRadix - 1)) : (unsigned int)kRadix;
      }
#pragma unroll
      for (int j = 0; j < kSortItems; ++j) {
        if (j < ipt) {
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
      }
      __syncthreads();
      // ---- per digit: exclusive offsets across warps, chunk base, advance the running base -----
      if (tid < kRadix) {
        unsigned int cnt = 0;
#pragma unroll
        for (int w = 0; w < kSortWarps; ++w) {
          const unsigned int c = s_wh[w][tid];
          s_wh[w][tid] = cnt;
          cnt += c;
        }
        const unsigned int b = s_hist[tid];
        s_cbase[tid] = b;
        s_hist[tid] = b + cnt;
      }
      __syncthreads();
      // ---- scatter -----------------------------------------------------------------------------
#pragma unroll
      for (int j = 0; j < kSortItems; ++j) {
        const unsigned int d = dig[j];
        if (j < ipt && d < (unsigned int)kRadix) {
          const unsigned int pos = s_cbase[d] + s_wh[warp][d] + rank[j];
          dk[pos] = key[j];
          dv[pos] = sv[wbase + j * 32 + lane];
        }
      }
      __syncthreads();
    }
    unsigned int* t;
    t = sk; sk = dk; dk = t;
    t = sv; sv = dv; dv = t;
  }
  // the result is in (sk, sv): shared A / B, or keys0 / keys1 after an even / odd number of passes.
  // ---- order runs of equal range bits by surfel index ------------------------------------------
  for (int i = tid; i + 1 < n; i += kSortThreads) {
    const unsigned int k = sk[i];
    if (sk[i + 1] == k && (i == 0 || sk[i - 1] != k)) {
      int e = i + 2;
      while (e < n && sk[e] == k) ++e;
      for (int p = i + 1; p < e; ++p) {              // insertion sort of sv[i, e) by surfel id
        const unsigned int v = sv[p];
        int q = p - 1;
        while (q >= i && sv[q] > v) { sv[q + 1] = sv[q]; --q; }
        sv[q + 1] = v;
      }
    }
  }
  if (in_smem || sk != keys0 + start) {
    __syncthreads();
    for (int i = tid; i < n; i += kSortThreads) { keys0[start + i] = sk[i]; vals0[start + i] = sv[i]; }
  }
}

}  // namespace

cudaError_t launch_tile_sort(uint32_t* keys0, uint32_t* keys1, uint32_t* vals0, uint32_t* vals1,
                             const unsigned int* ranges, const unsigned int* order, int nseg, cudaStream_t st) {
  if (nseg <= 0) return cudaSuccess;
  static bool attr_set = false;
  const size_t dyn = (size_t)4 * kSortSmemCap * sizeof(unsigned int);
  if (!attr_set) {
    cudaError_t e = cudaFuncSetAttribute(tile_sort_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dyn);
    if (e != cudaSuccess) return e;
    attr_set = true;
  }
  tile_sort_kernel<<<nseg, kSortThreads, dyn, st>>>(keys0, keys1, vals0, vals1, ranges, order);
  return cudaGetLastError();
}

}  // namespace lgs
