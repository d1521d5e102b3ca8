// K11: opacity prune + compaction of the map (first item; "opacity-based
// pruning", "alpha_min <= alpha_i").  A surfel is kept iff opacity >= alpha_min (NaN: dropped); the
// survivors keep their order; every per-surfel row (mu, q, s~, alpha, s, Adam moments m, v) moves with its surfel.
// Three kernels: per-block survivor counts; one-CTA exclusive scan of the block counts (+ the survivor total);
// order-preserving scatter (rank inside the block from warp ballots).
#include "lgs_internal.cuh"

namespace lgs {
namespace {

constexpr int kPruneThreads = 256;

struct PruneArgs {
  long long N;
  float alpha_min;
  const unsigned char* keep;   // optional keep flags [N] (lgs_compact): then alpha_min is not used
  const float* in[7];      // mean [N,3], quat [N,4], log_scale [N,2], opacity [N], scale [N,2], m [N,10], v [N,10]
  float* out[7];
  unsigned int* blk;       // per block: survivor count, then exclusive offset
  long long* n_out;
};

__device__ __forceinline__ bool keep_of(const PruneArgs& a, long long i) {
  if (i >= a.N) return false;
  return a.keep ? a.keep[i] != 0 : a.in[3][i] >= a.alpha_min;
}

__global__ void __launch_bounds__(kPruneThreads) prune_count_kernel(const PruneArgs a) {
  const long long i = (long long)blockIdx.x * kPruneThreads + threadIdx.x;
  const unsigned int c = (unsigned int)__syncthreads_count(keep_of(a, i));
  if (threadIdx.x == 0) a.blk[blockIdx.x] = c;
}

__global__ void __launch_bounds__(1024) prune_scan_kernel(unsigned int* blk, long long nb, long long* n_out) {
  __shared__ unsigned long long s_w[32];
  __shared__ unsigned long long s_carry;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  if (tid == 0) s_carry = 0;
  __syncthreads();
  for (long long base = 0; base < nb; base += 1024) {
    const long long b = base + tid;
    const unsigned long long c = (b < nb) ? blk[b] : 0ull;
    unsigned long long inc = c;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const unsigned long long v = __shfl_up_sync(0xffffffffu, inc, o);
      if (lane >= o) inc += v;
    }
    if (lane == 31) s_w[warp] = inc;
    __syncthreads();
    unsigned long long woff = 0, tot = 0;
    for (int w = 0; w < 32; ++w) { const unsigned long long x = s_w[w]; if (w < warp) woff += x; tot += x; }
    const unsigned long long carry = s_carry;
    if (b < nb) blk[b] = (unsigned int)(carry + woff + inc - c);       // exclusive offset (< N <= 2^24)
    __syncthreads();
    if (tid == 0) s_carry = carry + tot;
    __syncthreads();
  }
  if (tid == 0) *n_out = (long long)s_carry;
}

template <int W>
__device__ __forceinline__ void move_row(const float* in, float* out, long long src, long long dst) {
  if (!in || !out) return;
#pragma unroll
  for (int k = 0; k < W; ++k) out[(size_t)W * dst + k] = in[(size_t)W * src + k];
}

__global__ void __launch_bounds__(kPruneThreads) prune_scatter_kernel(const PruneArgs a) {
  __shared__ unsigned int s_w[kPruneThreads / 32];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const long long i = (long long)blockIdx.x * kPruneThreads + tid;
  const bool keep = keep_of(a, i);
  const unsigned int bal = __ballot_sync(0xffffffffu, keep);
  if (lane == 0) s_w[warp] = (unsigned int)__popc(bal);
  __syncthreads();
  unsigned int woff = 0;
#pragma unroll
  for (int w = 0; w < kPruneThreads / 32; ++w) woff += (w < warp) ? s_w[w] : 0u;
  if (!keep) return;
  const long long dst = (long long)a.blk[blockIdx.x] + woff + __popc(bal & ((1u << lane) - 1u));
  move_row<3>(a.in[0], a.out[0], i, dst);
  move_row<4>(a.in[1], a.out[1], i, dst);
  move_row<2>(a.in[2], a.out[2], i, dst);
  move_row<1>(a.in[3], a.out[3], i, dst);
  move_row<2>(a.in[4], a.out[4], i, dst);
  move_row<10>(a.in[5], a.out[5], i, dst);
  move_row<10>(a.in[6], a.out[6], i, dst);
}

}  // namespace

size_t prune_workspace_bytes(int64_t N) { return align_up((size_t)((N + kPruneThreads - 1) / kPruneThreads + 1) * 4); }

cudaError_t launch_prune(int64_t N, float alpha_min, const unsigned char* keep, const float* const in[7], float* const out[7], long long* n_out,
                         void* workspace, cudaStream_t st) {
  PruneArgs a;
  a.N = N; a.alpha_min = alpha_min; a.keep = keep;
  for (int k = 0; k < 7; ++k) { a.in[k] = in[k]; a.out[k] = out[k]; }
  a.blk = static_cast<unsigned int*>(workspace);
  a.n_out = n_out;
  const long long nb = (N + kPruneThreads - 1) / kPruneThreads;
  if (nb > 0) prune_count_kernel<<<(unsigned)nb, kPruneThreads, 0, st>>>(a);
  prune_scan_kernel<<<1, 1024, 0, st>>>(a.blk, nb, n_out);
  if (nb > 0) prune_scatter_kernel<<<(unsigned)nb, kPruneThreads, 0, st>>>(a);
  return cudaGetLastError();
}

}  // namespace lgs
