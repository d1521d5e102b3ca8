// K9: optimiser step that closes the mapping iteration.
//   Theta = {mu, q, s~, alpha}, s~ = log s;
//   L_scale = sum_i max(0, max(s_i0, s_i1) - s_max) (Eq. 12) enters with weight lambda_s (Eq. 13);
//   the update rule is Adam with bias correction (reading R21: the paper names no optimiser).
// One thread per surfel: 40 B of parameters, 40 B of gradients and 80 B of moments in, 48 B of parameters
// (+ the activated scale) and 80 B of moments out -- a streaming kernel bound by HBM bandwidth
// (288 B per surfel).
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
  float inv_bc1, inv_bc2;      // 1 / (1 - b1^t), 1 / (1 - b2^t)
  float lambda_s, s_max, alpha_lo, alpha_hi;
  float* loss_scale;
};

__device__ __forceinline__ float adam1(float theta, float g, float& m, float& v, float lr, const AdamArgs& a) {
  m = a.b1 * m + (1.0f - a.b1) * g;
  v = a.b2 * v + (1.0f - a.b2) * g * g;
  const float mh = m * a.inv_bc1, vh = v * a.inv_bc2;
  return theta - lr * mh / (sqrtf(vh) + a.eps);
}

__global__ void __launch_bounds__(256) adam_step_kernel(const AdamArgs a) {
  __shared__ float s_red[8];
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  float lsc = 0.f;
  if (i < a.N) {
    // ---- loads: everything of the surfel up front ------------------------------------------------
    float th[10], g[10], m[10], v[10];
    th[0] = a.mean[3 * i]; th[1] = a.mean[3 * i + 1]; th[2] = a.mean[3 * i + 2];
    const float4 q = reinterpret_cast<const float4*>(a.quat)[i];
    th[3] = q.x; th[4] = q.y; th[5] = q.z; th[6] = q.w;
    const float2 ls = reinterpret_cast<const float2*>(a.log_scale)[i];
    th[7] = ls.x; th[8] = ls.y;
    th[9] = a.opacity[i];
    g[0] = a.g_mean[3 * i]; g[1] = a.g_mean[3 * i + 1]; g[2] = a.g_mean[3 * i + 2];
    const float4 gq = reinterpret_cast<const float4*>(a.g_quat)[i];
    g[3] = gq.x; g[4] = gq.y; g[5] = gq.z; g[6] = gq.w;
    const float2 gs = reinterpret_cast<const float2*>(a.g_scale)[i];
    g[9] = a.g_opacity[i];
    const float2* mr = reinterpret_cast<const float2*>(a.m + 10 * i);
    const float2* vr = reinterpret_cast<const float2*>(a.v + 10 * i);
#pragma unroll
    for (int k = 0; k < 5; ++k) {
      const float2 mm = mr[k], vv = vr[k];
      m[2 * k] = mm.x; m[2 * k + 1] = mm.y; v[2 * k] = vv.x; v[2 * k + 1] = vv.y;
    }
    // ---- Eq. 12 and the chain rule of s = exp(s~) ---------------------------------------------------
    const float s0 = expf(th[7]), s1 = expf(th[8]);
    const float top = fmaxf(s0, s1);
    float r0 = 0.f, r1 = 0.f;
    if (top - a.s_max > 0.f) {
      lsc = top - a.s_max;
      if (s0 > s1) r0 = 1.f; else if (s1 > s0) r1 = 1.f; else { r0 = 0.5f; r1 = 0.5f; }
    }
    g[7] = s0 * (gs.x + a.lambda_s * r0);
    g[8] = s1 * (gs.y + a.lambda_s * r1);
    // ---- Adam ---------------------------------------------------------------------------------------
#pragma unroll
    for (int k = 0; k < 10; ++k) th[k] = adam1(th[k], g[k], m[k], v[k], a.lr[k < 3 ? 0 : (k < 7 ? 1 : (k < 9 ? 2 : 3))], a);
    th[9] = fminf(fmaxf(th[9], a.alpha_lo), a.alpha_hi);
    // ---- stores -------------------------------------------------------------------------------------
    a.mean[3 * i] = th[0]; a.mean[3 * i + 1] = th[1]; a.mean[3 * i + 2] = th[2];
    reinterpret_cast<float4*>(a.quat)[i] = make_float4(th[3], th[4], th[5], th[6]);
    reinterpret_cast<float2*>(a.log_scale)[i] = make_float2(th[7], th[8]);
    reinterpret_cast<float2*>(a.scale)[i] = make_float2(expf(th[7]), expf(th[8]));
    a.opacity[i] = th[9];
    float2* mw = reinterpret_cast<float2*>(a.m + 10 * i);
    float2* vw = reinterpret_cast<float2*>(a.v + 10 * i);
#pragma unroll
    for (int k = 0; k < 5; ++k) { mw[k] = make_float2(m[2 * k], m[2 * k + 1]); vw[k] = make_float2(v[2 * k], v[2 * k + 1]); }
  }
  // ---- L_scale before the step: block reduction, one atomic per block ------------------------------
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) lsc += __shfl_xor_sync(0xffffffffu, lsc, o);
  if ((threadIdx.x & 31) == 0) s_red[threadIdx.x >> 5] = lsc;
  __syncthreads();
  if (threadIdx.x == 0) {
    float t = 0.f;
    for (int w = 0; w < 8; ++w) t += s_red[w];
    if (t != 0.f) atomicAdd(a.loss_scale, t);
  }
}

}  // namespace

cudaError_t launch_adam(int64_t N, float* mean, float* quat, float* log_scale, float* opacity, float* scale,
                        const float* g_mean, const float* g_quat, const float* g_scale, const float* g_opacity,
                        float* m, float* v, const lgs_adam& h, float* loss_scale, cudaStream_t st) {
  cudaError_t e = cudaMemsetAsync(loss_scale, 0, sizeof(float), st);
  if (e != cudaSuccess || N <= 0) return e;
  AdamArgs a;
  a.N = N;
  a.mean = mean; a.quat = quat; a.log_scale = log_scale; a.opacity = opacity; a.scale = scale;
  a.g_mean = g_mean; a.g_quat = g_quat; a.g_scale = g_scale; a.g_opacity = g_opacity;
  a.m = m; a.v = v;
  a.lr[0] = h.lr_mean; a.lr[1] = h.lr_quat; a.lr[2] = h.lr_scale; a.lr[3] = h.lr_opacity;
  a.b1 = h.beta1; a.b2 = h.beta2; a.eps = h.eps;
  // bias corrections in double on the host (t can be large)
  a.inv_bc1 = (float)(1.0 / (1.0 - std::pow((double)h.beta1, (double)h.step)));
  a.inv_bc2 = (float)(1.0 / (1.0 - std::pow((double)h.beta2, (double)h.step)));
  a.lambda_s = h.lambda_s; a.s_max = h.s_max; a.alpha_lo = h.alpha_lo; a.alpha_hi = h.alpha_hi;
  a.loss_scale = loss_scale;
  adam_step_kernel<<<(unsigned)((N + 255) / 256), 256, 0, st>>>(a);
  return cudaGetLastError();
}

}  // namespace lgs
