// Micro-benchmarks behind the roofline denominators ("the builder must confirm ... both rates with
// an FFMA and a MUFU.EX2 micro-benchmark and record the sustained clock").
//   LGS_MB_FFMA      FP32 issue peak: dependent FFMA chains, 8 independent accumulators per thread, 64 warps per SM
//   LGS_MB_MUFU_EX2  SFU peak: ex2.approx.ftz.f32 chains, same shape
//   LGS_MB_RED_F32 / LGS_MB_RED_F32X4  throughput of the backward's scatter-add into 64-byte per-surfel rows:
//                    13 scalar red.global.add.f32 per row visit against 4 red.global.add.v4.f32 (sm_90+)
// lgs_microbench times its own launches with CUDA events and synchronises: a measurement aid, not part of the path.
#include "lgs_internal.cuh"

namespace lgs {
namespace {

constexpr int kMbThreads = 1024;
constexpr int kMbIters = 4096;
constexpr int kMbAcc = 8;

__global__ void __launch_bounds__(kMbThreads) mb_ffma_kernel(float* out, float a, float b) {
  float x[kMbAcc];
#pragma unroll
  for (int k = 0; k < kMbAcc; ++k) x[k] = (float)(threadIdx.x + k);
  for (int it = 0; it < kMbIters; ++it) {
#pragma unroll
    for (int k = 0; k < kMbAcc; ++k) x[k] = __fmaf_rn(x[k], a, b);
  }
  float s = 0.f;
#pragma unroll
  for (int k = 0; k < kMbAcc; ++k) s += x[k];
  if (s == 123.456f) out[0] = s;      // keeps the chains alive; practically never true
}

__global__ void __launch_bounds__(kMbThreads) mb_mufu_kernel(float* out, float a) {
  float x[kMbAcc];
#pragma unroll
  for (int k = 0; k < kMbAcc; ++k) x[k] = a * (float)(threadIdx.x + k);
  for (int it = 0; it < kMbIters; ++it) {
#pragma unroll
    for (int k = 0; k < kMbAcc; ++k) asm volatile("ex2.approx.ftz.f32 %0, %0;" : "+f"(x[k]));
  }
  float s = 0.f;
#pragma unroll
  for (int k = 0; k < kMbAcc; ++k) s += x[k];
  if (s == 123.456f) out[0] = s;
}

// Every thread visits `visits` pseudo-random 64-byte rows of `rows` and adds 13 (scalar) or 16 (4 x v4) floats.
// share: groups of `share` consecutive lanes visit the same row (1 = every lane its own row).
template <bool kVec>
__global__ void __launch_bounds__(256) mb_red_kernel(float* buf, unsigned int rows, int visits, int share) {
  const unsigned int t = blockIdx.x * blockDim.x + threadIdx.x;
  unsigned int h = (t / (unsigned int)share) * 2654435761u + 12345u;
  for (int it = 0; it < visits; ++it) {
    h = h * 1664525u + 1013904223u;
    float* row = buf + (size_t)((h >> 8) % rows) * 16;
    const float v = (float)(it & 3);
    if (kVec) {
#pragma unroll
      for (int k = 0; k < 4; ++k)
        asm volatile("red.global.add.v4.f32 [%0], {%1, %1, %1, %1};" ::"l"(row + 4 * k), "f"(v) : "memory");
    } else {
#pragma unroll
      for (int k = 0; k < 13; ++k) atomicAdd(row + k, v);
    }
  }
}

}  // namespace
}  // namespace lgs

using namespace lgs;

extern "C" lgs_status lgs_microbench(int which, void* scratch, size_t scratch_bytes, int param, double* rate_per_s,
                                     float* ms_out, lgs_stream stream) {
  if (!rate_per_s || !scratch || scratch_bytes < 64) return LGS_ERR_INVALID_ARG;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  cudaEvent_t e0, e1;
  if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) return LGS_ERR_CUDA;
  const int sms = sm_count();
  double work = 0.0;
  float best = 1e30f;
  for (int rep = 0; rep < 6; ++rep) {          // rep 0 warms up (clocks, instruction cache)
    cudaEventRecord(e0, st);
    switch (which) {
      case LGS_MB_FFMA:
        mb_ffma_kernel<<<sms * 2, kMbThreads, 0, st>>>(static_cast<float*>(scratch), 1.0000001f, 1e-9f);
        work = (double)sms * 2 * kMbThreads * (double)kMbIters * kMbAcc;
        break;
      case LGS_MB_MUFU_EX2:
        mb_mufu_kernel<<<sms * 2, kMbThreads, 0, st>>>(static_cast<float*>(scratch), -1e-3f);
        work = (double)sms * 2 * kMbThreads * (double)kMbIters * kMbAcc;
        break;
      case LGS_MB_RED_F32:
      case LGS_MB_RED_F32X4: {
        const unsigned int rows = (unsigned int)(scratch_bytes / 64);
        const int visits = 64, share = param > 0 ? param : 1;
        if (which == LGS_MB_RED_F32) mb_red_kernel<false><<<sms * 8, 256, 0, st>>>(static_cast<float*>(scratch), rows, visits, share);
        else mb_red_kernel<true><<<sms * 8, 256, 0, st>>>(static_cast<float*>(scratch), rows, visits, share);
        work = (double)sms * 8 * 256 * visits;     // row visits
        break;
      }
      default:
        cudaEventDestroy(e0); cudaEventDestroy(e1);
        return LGS_ERR_INVALID_ARG;
    }
    cudaEventRecord(e1, st);
    if (cudaEventSynchronize(e1) != cudaSuccess) { cudaEventDestroy(e0); cudaEventDestroy(e1); return LGS_ERR_CUDA; }
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    if (rep > 0 && ms < best) best = ms;
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  if (cudaGetLastError() != cudaSuccess) return LGS_ERR_CUDA;
  *rate_per_s = work / ((double)best * 1e-3);
  if (ms_out) *ms_out = best;
  return LGS_OK;
}
