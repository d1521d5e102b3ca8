// K11: opacity prune + compaction of the map (first item; "opacity-based
// pruning", "alpha_min <= alpha_i").  A surfel is kept iff opacity >= alpha_min (NaN: dropped); the
// survivors keep their order; every per-surfel row (mu, q, s~, alpha, s, Adam moments m, v) moves with its surfel.
// Three kernels (overlapped with programmatic dependent launch): per-block survivor counts; one-CTA exclusive scan of the
// block counts (+ the survivor total); order-preserving scatter: rank inside the block from warp ballots, every array's rows
// cross shared memory so that global memory sees a coalesced read of the block's chunk and a coalesced write of the
// survivors' rows (the survivors of a block are contiguous in the output).
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
  asm volatile("griddepcontrol.launch_dependents;");     // the scan CTA becomes resident and waits for the counts
  const long long i = (long long)blockIdx.x * kPruneThreads + threadIdx.x;
  const unsigned int c = (unsigned int)__syncthreads_count(keep_of(a, i));
  if (threadIdx.x == 0) a.blk[blockIdx.x] = c;
}

__global__ void __launch_bounds__(1024) prune_scan_kernel(unsigned int* blk, long long nb, long long* n_out) {
  __shared__ unsigned long long s_w[32];
  __shared__ unsigned long long s_carry;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  // launched with programmatic stream serialisation behind the count kernel; lets the scatter kernel in at once
  asm volatile("griddepcontrol.wait;" ::: "memory");
  asm volatile("griddepcontrol.launch_dependents;");
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

// The CTA's rows of one array cross shared memory: a coalesced (16-byte) read of the CTA's contiguous input chunk, then a
// coalesced write of the survivors' rows, which are contiguous in the output ([base, base + cnt) rows).
template <int W>
__device__ __forceinline__ void move_rows(const float* __restrict__ in, float* __restrict__ out, long long i0, int nb,
                                          long long base, int cnt, const unsigned short* s_src, float* s_buf, int tid) {
  if (!in || !out) return;                   // (uniform)
  const float* src = in + (size_t)W * i0;    // 1 KiB-aligned relative to the array base (i0 is a multiple of 256)
  const int n = W * nb, n4 = n >> 2;
  for (int k = tid; k < n4; k += kPruneThreads) reinterpret_cast<float4*>(s_buf)[k] = reinterpret_cast<const float4*>(src)[k];
  for (int k = (n4 << 2) + tid; k < n; k += kPruneThreads) s_buf[k] = src[k];
  __syncthreads();
  float* dst = out + (size_t)W * base;
  for (int e = tid; e < W * cnt; e += kPruneThreads) {
    const int r = e / W, c = e - r * W;
    dst[e] = s_buf[(int)s_src[r] * W + c];
  }
  __syncthreads();
}

__global__ void __launch_bounds__(kPruneThreads) prune_scatter_kernel(const PruneArgs a) {
  __shared__ unsigned int s_w[kPruneThreads / 32];
  __shared__ unsigned short s_src[kPruneThreads];
  __shared__ __align__(16) float s_buf[10 * kPruneThreads];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const long long i0 = (long long)blockIdx.x * kPruneThreads;
  const long long i = i0 + tid;
  const bool keep = keep_of(a, i);
  const unsigned int bal = __ballot_sync(0xffffffffu, keep);
  if (lane == 0) s_w[warp] = (unsigned int)__popc(bal);
  __syncthreads();
  unsigned int woff = 0, cnt = 0;
#pragma unroll
  for (int w = 0; w < kPruneThreads / 32; ++w) { const unsigned int x = s_w[w]; if (w < warp) woff += x; cnt += x; }
  if (keep) s_src[woff + (unsigned int)__popc(bal & ((1u << lane) - 1u))] = (unsigned short)tid;
  // launched beside the scan kernel (which computes this block's output offset): everything above needs only the inputs
  asm volatile("griddepcontrol.wait;" ::: "memory");
  __syncthreads();
  const long long base = (long long)a.blk[blockIdx.x];
  const int nb = (int)min((long long)kPruneThreads, a.N - i0);
  move_rows<3>(a.in[0], a.out[0], i0, nb, base, (int)cnt, s_src, s_buf, tid);
  move_rows<4>(a.in[1], a.out[1], i0, nb, base, (int)cnt, s_src, s_buf, tid);
  move_rows<2>(a.in[2], a.out[2], i0, nb, base, (int)cnt, s_src, s_buf, tid);
  move_rows<1>(a.in[3], a.out[3], i0, nb, base, (int)cnt, s_src, s_buf, tid);
  move_rows<2>(a.in[4], a.out[4], i0, nb, base, (int)cnt, s_src, s_buf, tid);
  move_rows<10>(a.in[5], a.out[5], i0, nb, base, (int)cnt, s_src, s_buf, tid);
  move_rows<10>(a.in[6], a.out[6], i0, nb, base, (int)cnt, s_src, s_buf, tid);
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
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  unsigned int* blk = a.blk;
  e = launch_pdl(prune_scan_kernel, dim3(1), dim3(1024), 0, st, blk, (long long)nb, n_out);
  if (e != cudaSuccess) return e;
  if (nb > 0) e = launch_pdl(prune_scatter_kernel, dim3((unsigned)nb), dim3(kPruneThreads), 0, st, a);
  return e;
}

}  // namespace lgs
