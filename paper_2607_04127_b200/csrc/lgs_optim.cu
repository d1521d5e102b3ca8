// K9: optimiser step that closes the mapping iteration.
//   Theta = {mu, q, s~, alpha}, s~ = log s;
//   L_scale = sum_i max(0, max(s_i0, s_i1) - s_max) (Eq. 12) enters with weight lambda_s (Eq. 13);
//   the update rule is Adam with bias correction (reading R21: the paper names no optimiser).
// One thread per surfel, one CTA per kAdamThreads = 256 surfels (64 / 128 / 256 measure the same 21.4-22 us): 40 B of parameters, 40 B of gradients and 80 B of moments in,
// 48 B of parameters (+ the activated scale) and 80 B of moments out -- a streaming kernel bound by HBM bandwidth
// (288 B per surfel).  The 12- and 40-byte rows (mu, g_mu, m, v) cross shared memory so
// that global memory only sees coalesced 16-byte accesses.
#include <cmath>
#include "lgs_internal.cuh"

namespace lgs {
namespace {

struct AdamArgs {
  long long N;
  float* mean; float* quat; float* log_scale; float* opacity; float* scale;
  const float* g_mean; const float* g_quat; const float* g_scale; const float* g_opacity;
  float* m; float* v;
  float lr[4];                 // mu, q, s~, alpha
  float b1, b2, eps;
  float inv_bc1, inv_bc2;      // 1 / (1 - b1^t), 1 / (1 - b2^t)  (t from the host)
  const int* step_dev;         // if not NULL: t is read on the device and the two factors are computed here
  float lambda_s, s_max, alpha_lo, alpha_hi;
  float* loss_scale;
};

__device__ __forceinline__ float adam1(float theta, float g, float& m, float& v, float lr, const AdamArgs& a,
                                       float inv_bc1, float inv_bc2) {
  m = a.b1 * m + (1.0f - a.b1) * g;
  v = a.b2 * v + (1.0f - a.b2) * g * g;
  const float mh = m * inv_bc1, vh = v * inv_bc2;
  return theta - lr * mh / (sqrtf(vh) + a.eps);
}

// Coalesced 16-byte copies between a contiguous global range [0, count) floats of this CTA and shared memory
// (the rows of a surfel are 12 / 40 bytes: per-thread row accesses would touch every line five times).
#ifndef LGS_ADAM_THREADS
#define LGS_ADAM_THREADS 256
#endif
constexpr int kAdamThreads = LGS_ADAM_THREADS;      // surfels per CTA

__device__ __forceinline__ void cta_load(float* dst, const float* src, int count, int tid) {
  const int n4 = count >> 2;
  for (int k = tid; k < n4; k += kAdamThreads) reinterpret_cast<float4*>(dst)[k] = reinterpret_cast<const float4*>(src)[k];
  for (int k = (n4 << 2) + tid; k < count; k += kAdamThreads) dst[k] = src[k];
}
__device__ __forceinline__ void cta_store(float* dst, const float* src, int count, int tid) {
  const int n4 = count >> 2;
  for (int k = tid; k < n4; k += kAdamThreads) reinterpret_cast<float4*>(dst)[k] = reinterpret_cast<const float4*>(src)[k];
  for (int k = (n4 << 2) + tid; k < count; k += kAdamThreads) dst[k] = src[k];
}

// Zeroes the L_scale accumulator; the step kernel is launched beside it (programmatic dependent launch) and waits only
// before its one atomic per block.
__global__ void adam_zero_kernel(float* loss_scale) {
  asm volatile("griddepcontrol.launch_dependents;");
  *loss_scale = 0.f;
}

__global__ void __launch_bounds__(kAdamThreads) adam_step_kernel(const AdamArgs a) {
  __shared__ __align__(16) float s_m[10 * kAdamThreads], s_v[10 * kAdamThreads], s_mean[3 * kAdamThreads], s_gmean[3 * kAdamThreads];
  __shared__ float s_red[kAdamThreads / 32];
  __shared__ float s_bc[2];
  const int tid = threadIdx.x;
  if (tid == 0) {
    s_bc[0] = a.inv_bc1; s_bc[1] = a.inv_bc2;
    if (a.step_dev) {                      // same fp64 expression as the host path of launch_adam
      const double t = (double)max(*a.step_dev, 1);
      s_bc[0] = (float)(1.0 / (1.0 - pow((double)a.b1, t)));
      s_bc[1] = (float)(1.0 / (1.0 - pow((double)a.b2, t)));
    }
  }
  const long long i0 = (long long)blockIdx.x * kAdamThreads;
  const int nb = (int)min((long long)kAdamThreads, a.N - i0);     // surfels of this CTA
  const long long i = i0 + tid;
  // ---- loads: the CTA's rows of the moments and of mu, g_mu through shared memory (16-byte, coalesced) ----------
  cta_load(s_m, a.m + 10 * i0, 10 * nb, tid);
  cta_load(s_v, a.v + 10 * i0, 10 * nb, tid);
  cta_load(s_mean, a.mean + 3 * i0, 3 * nb, tid);
  cta_load(s_gmean, a.g_mean + 3 * i0, 3 * nb, tid);
  float lsc = 0.f;
  float th[10], g[10];
  if (tid < nb) {
    const float4 q = reinterpret_cast<const float4*>(a.quat)[i];
    th[3] = q.x; th[4] = q.y; th[5] = q.z; th[6] = q.w;
    const float2 ls = reinterpret_cast<const float2*>(a.log_scale)[i];
    th[7] = ls.x; th[8] = ls.y;
    th[9] = a.opacity[i];
    const float4 gq = reinterpret_cast<const float4*>(a.g_quat)[i];
    g[3] = gq.x; g[4] = gq.y; g[5] = gq.z; g[6] = gq.w;
    const float2 gs = reinterpret_cast<const float2*>(a.g_scale)[i];
    g[7] = gs.x; g[8] = gs.y;
    g[9] = a.g_opacity[i];
  }
  __syncthreads();
  if (tid < nb) {
    float m[10], v[10];
#pragma unroll
    for (int k = 0; k < 10; ++k) { m[k] = s_m[10 * tid + k]; v[k] = s_v[10 * tid + k]; }
#pragma unroll
    for (int k = 0; k < 3; ++k) { th[k] = s_mean[3 * tid + k]; g[k] = s_gmean[3 * tid + k]; }
    // ---- Eq. 12 and the chain rule of s = exp(s~) ---------------------------------------------------
    const float s0 = expf(th[7]), s1 = expf(th[8]);
    const float top = fmaxf(s0, s1);
    float r0 = 0.f, r1 = 0.f;
    if (top - a.s_max > 0.f) {
      lsc = top - a.s_max;
      if (s0 > s1) r0 = 1.f; else if (s1 > s0) r1 = 1.f; else { r0 = 0.5f; r1 = 0.5f; }
    }
    g[7] = s0 * (g[7] + a.lambda_s * r0);
    g[8] = s1 * (g[8] + a.lambda_s * r1);
    // ---- Adam ---------------------------------------------------------------------------------------
    const float inv_bc1 = s_bc[0], inv_bc2 = s_bc[1];      // (written before the barrier above)
#pragma unroll
    for (int k = 0; k < 10; ++k)
      th[k] = adam1(th[k], g[k], m[k], v[k], a.lr[k < 3 ? 0 : (k < 7 ? 1 : (k < 9 ? 2 : 3))], a, inv_bc1, inv_bc2);
    th[9] = fminf(fmaxf(th[9], a.alpha_lo), a.alpha_hi);
    // ---- stores -------------------------------------------------------------------------------------
#pragma unroll
    for (int k = 0; k < 10; ++k) { s_m[10 * tid + k] = m[k]; s_v[10 * tid + k] = v[k]; }
#pragma unroll
    for (int k = 0; k < 3; ++k) s_mean[3 * tid + k] = th[k];
    reinterpret_cast<float4*>(a.quat)[i] = make_float4(th[3], th[4], th[5], th[6]);
    reinterpret_cast<float2*>(a.log_scale)[i] = make_float2(th[7], th[8]);
    reinterpret_cast<float2*>(a.scale)[i] = make_float2(expf(th[7]), expf(th[8]));
    a.opacity[i] = th[9];
  }
  // ---- L_scale before the step: block reduction, one atomic per block ------------------------------
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) lsc += __shfl_xor_sync(0xffffffffu, lsc, o);
  if ((tid & 31) == 0) s_red[tid >> 5] = lsc;
  __syncthreads();
  cta_store(a.m + 10 * i0, s_m, 10 * nb, tid);
  cta_store(a.v + 10 * i0, s_v, 10 * nb, tid);
  cta_store(a.mean + 3 * i0, s_mean, 3 * nb, tid);
  asm volatile("griddepcontrol.wait;" ::: "memory");     // the accumulator is zero (every path of the grid gets here)
  if (tid == 0) {
    float t = 0.f;
    for (int w = 0; w < kAdamThreads / 32; ++w) t += s_red[w];
    if (t != 0.f) atomicAdd(a.loss_scale, t);
  }
}

}  // namespace

cudaError_t launch_adam(int64_t N, float* mean, float* quat, float* log_scale, float* opacity, float* scale,
                        const float* g_mean, const float* g_quat, const float* g_scale, const float* g_opacity,
                        float* m, float* v, const lgs_adam& h, float* loss_scale, cudaStream_t st) {
  adam_zero_kernel<<<1, 1, 0, st>>>(loss_scale);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess || N <= 0) return e;
  AdamArgs a;
  a.N = N;
  a.mean = mean; a.quat = quat; a.log_scale = log_scale; a.opacity = opacity; a.scale = scale;
  a.g_mean = g_mean; a.g_quat = g_quat; a.g_scale = g_scale; a.g_opacity = g_opacity;
  a.m = m; a.v = v;
  a.lr[0] = h.lr_mean; a.lr[1] = h.lr_quat; a.lr[2] = h.lr_scale; a.lr[3] = h.lr_opacity;
  a.b1 = h.beta1; a.b2 = h.beta2; a.eps = h.eps;
  // bias corrections in double on the host (t can be large)
  const double t = (double)(h.step > 0 ? h.step : 1);
  a.inv_bc1 = (float)(1.0 / (1.0 - std::pow((double)h.beta1, t)));
  a.inv_bc2 = (float)(1.0 / (1.0 - std::pow((double)h.beta2, t)));
  a.step_dev = h.step_device;
  a.lambda_s = h.lambda_s; a.s_max = h.s_max; a.alpha_lo = h.alpha_lo; a.alpha_hi = h.alpha_hi;
  a.loss_scale = loss_scale;
  return launch_pdl(adam_step_kernel, dim3((unsigned)((N + kAdamThreads - 1) / kAdamThreads)), dim3(kAdamThreads), 0, st, a);
}

}  // namespace lgs
