// K6: image-space loss stage (step S6 of SURVEY.md 8(a)).
//   L_depth  masked L1 range loss            (Eq. 10 left,  PAPER.md:131; valid pixels PAPER.md:127)
//   L_ng     cosine loss vs N_g-icp on M_N   (Eq. 11 first term)
//   L_ns     cosine loss vs N_surf computed from the rendered range (Eq. 11 second term),
//            central differences of X = D^ d over the 4-neighbourhood (columns wrap at the seam),
//            gradient flowing into D^ of the neighbours unless detach_surf (reading R11)
//   L_alpha  positive-only BCE(A^, 1) = -log(A^ + eps) on M_D  (Eq. 10 right; lgs_loss_mapping only)
//   L = L_depth + lambda_alpha L_alpha + lambda_n (lambda_ng L_ng + lambda_ns L_ns)      (Eq. 13, image side)
// Two kernels: (1) count |Omega_M|, |Omega_N| (per-block partial counts: no counter to clear beforehand),
// clear the gradient images and fill the beam table (fp64 sincos once per column / row instead of per
// pixel and neighbour); (2) everything else.  Kernel (1) is launched with programmatic stream serialisation:
// its reads of the targets, the counting and the fp64 sincos run beside the tail of whatever precedes it in the
// stream; its writes wait for that to complete (a previous loss call on the same buffers may still be running);
// kernel (2) is launched normally.
#include "lgs_internal.cuh"

namespace lgs {
namespace {

constexpr double kPi = 3.14159265358979323846;

struct LossWs {
  unsigned int nS, done, pad0, pad1;
  double Ld, Lng, Lns, La;
};
constexpr int kLossHdr = 256;        // bytes of LossWs slot; then the beam table, then the per-block counts

struct LossArgs {
  int H, W;
  double elev_max, dphi, dth;
  const float* range; const float* normal; const float* target; const float* tnormal; const uint8_t* keep;
  const float* alpha;              // A^ (read only when lambda_alpha != 0)
  float lambda_alpha, alpha_eps;   // Eq. 10 right / Eq. 13; lambda_alpha = 0: no opacity term, loss has 4 entries
  int n_loss;                      // 4 (lgs_loss_range_normal) or 5 (lgs_loss_mapping)
  float lambda_n, lambda_ng, lambda_ns;
  int detach;
  LossWs* ws;
  double* beams;                   // [2W + 2H]: cos phi, sin phi per column; cos theta, sin theta per row
  uint2* blk_cnt;                  // per block of the count kernel: {|Omega_M|, |Omega_N|} of its pixels
  float* loss; float* gD; float* gA; float* gN;
};

__device__ __forceinline__ bool in_M(const LossArgs& a, size_t px) {
  return a.target[px] > 0.f && (!a.keep || a.keep[px] != 0);
}

// Beam-table entry k (k < W: cos / sin of column k's azimuth; else of row k - W's elevation).
__device__ __forceinline__ void beam_entry(const LossArgs& a, size_t k, double* cs, double* sn) {
  if (k < (size_t)a.W) sincos(-kPi + ((double)k + 0.5) * a.dphi, sn, cs);
  else sincos(a.elev_max - ((double)(k - a.W) + 0.5) * a.dth, sn, cs);
}
__device__ __forceinline__ void beam_store(const LossArgs& a, size_t k, double cs, double sn) {
  if (k < (size_t)a.W) { a.beams[k] = cs; a.beams[a.W + k] = sn; }
  else { const size_t j = k - a.W; a.beams[2 * a.W + j] = cs; a.beams[2 * a.W + a.H + j] = sn; }
}

// Launched with programmatic stream serialisation: the grid may become resident while kernels that precede it in the
// stream still run -- the forward composite (which lets its dependents in early), but also the loss_grad_kernel of a
// PREVIOUS loss call on the same workspace and gradient images, which is still adding into gD and the loss sums after
// its launch_dependents.  So everything above griddepcontrol.wait only READS the caller's inputs (targets, mask) and
// computes in registers; every write (gradient images, beam table, block counts, counters) comes after it, when all
// earlier work in the stream has completed and flushed.  The wait is on every path, so "this grid completed" still
// implies "everything before it completed" for loss_grad_kernel, which is launched in plain stream order behind it.
__global__ void __launch_bounds__(256) loss_count_kernel(const LossArgs a) {
  const size_t HW = (size_t)a.H * a.W;
  const size_t px = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  const size_t nb = (size_t)(a.W + a.H), stride = (size_t)gridDim.x * blockDim.x;
  double cs0 = 0.0, sn0 = 0.0;
  if (px < nb) beam_entry(a, px, &cs0, &sn0);
  bool m = false, n = false;
  if (px < HW) {
    m = in_M(a, px);
    if (m && a.tnormal) {
      const float x = a.tnormal[px], y = a.tnormal[HW + px], z = a.tnormal[2 * HW + px];
      n = (x * x + y * y + z * z) > 0.f;
    }
  }
  const unsigned int cm = __syncthreads_count(m), cn = __syncthreads_count(n);
  asm volatile("griddepcontrol.wait;" ::: "memory");
  if (px < nb) beam_store(a, px, cs0, sn0);
  for (size_t k = px + stride; k < nb; k += stride) {       // only a 1-row or 1-column image has more entries than threads
    double cs, sn;
    beam_entry(a, k, &cs, &sn);
    beam_store(a, k, cs, sn);
  }
  if (px < HW) {
    a.gD[px] = 0.f;
    a.gA[px] = 0.f;
  }
  if (threadIdx.x == 0) {
    a.blk_cnt[blockIdx.x] = make_uint2(cm, cn);
    if (blockIdx.x == 0) { a.ws->nS = 0u; a.ws->done = 0u; a.ws->Ld = 0.0; a.ws->Lng = 0.0; a.ws->Lns = 0.0; a.ws->La = 0.0; }
  }
}

__device__ __forceinline__ void beam_dir(const LossArgs& a, int j, int i, float* d) {
  const double cp = a.beams[i], sp = a.beams[a.W + i], ct = a.beams[2 * a.W + j], st = a.beams[2 * a.W + a.H + j];
  d[0] = (float)(ct * cp); d[1] = (float)(ct * sp); d[2] = (float)st;
}

__global__ void __launch_bounds__(256) loss_grad_kernel(const LossArgs a) {
  __shared__ double s_red[4][8];
  __shared__ unsigned int s_cnt[8];
  const int H = a.H, W = a.W;
  const size_t HW = (size_t)H * W;
  const size_t px = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  // the backward's first kernel (it clears the partial sums) may run beside this small grid
  asm volatile("griddepcontrol.launch_dependents;");
  // every load of the pixel and its 4-neighbourhood is issued up front (one round trip, not a chain), together
  // with the count kernel's per-block counts
  const bool inb = px < HW;
  const int j = inb ? (int)(px / W) : 0, i = inb ? (int)(px % W) : 0;
  const bool inner = j >= 1 && j + 1 < H;
  const int ip = (i + 1 == W) ? 0 : i + 1, im = (i == 0) ? W - 1 : i - 1;
  const size_t p0 = inb ? px : 0;
  const size_t pe = (size_t)j * W + ip, pw = (size_t)j * W + im, pu = inner ? p0 - W : p0, pd = inner ? p0 + W : p0;
  const bool m0 = inb && in_M(a, p0), mE = in_M(a, pe), mW = in_M(a, pw), mU = in_M(a, pu), mD = in_M(a, pd);
  const float r0 = a.range[p0], re = a.range[pe], rw = a.range[pw], ru = a.range[pu], rd = a.range[pd];
  const float t0 = a.target[p0];
  // |Omega_M|, |Omega_N|: sum of the count kernel's per-block counts (same grid)
  __shared__ unsigned int s_n[2];
  if (threadIdx.x < 2) s_n[threadIdx.x] = 0u;
  __syncthreads();
  {
    unsigned int cm = 0, cn = 0;
    for (unsigned int b = threadIdx.x; b < gridDim.x; b += blockDim.x) { const uint2 c = a.blk_cnt[b]; cm += c.x; cn += c.y; }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) { cm += __shfl_xor_sync(0xffffffffu, cm, o); cn += __shfl_xor_sync(0xffffffffu, cn, o); }
    if ((threadIdx.x & 31) == 0) { if (cm) atomicAdd(&s_n[0], cm); if (cn) atomicAdd(&s_n[1], cn); }
  }
  __syncthreads();
  const unsigned int nM = s_n[0], nN = s_n[1];
  double ld = 0.0, lng = 0.0, lns = 0.0, la = 0.0;
  unsigned int ns_cnt = 0;
  if (inb && nM > 0) {
    float gn[3] = {0.f, 0.f, 0.f};
    if (m0) {
      const float invM = 1.0f / (float)nM;
      const float e = r0 - t0;
      ld = fabsf(e);
      const float sg = (e > 0.f) ? 1.f : ((e < 0.f) ? -1.f : 0.f);
      if (sg != 0.f) atomicAdd(&a.gD[px], sg * invM);
      if (a.lambda_alpha != 0.f) {
        const float ae = a.alpha[px] + a.alpha_eps;
        la = -log((double)ae);
        a.gA[px] = -a.lambda_alpha * invM / ae;      // gA was cleared by the count kernel; only this thread writes it
      }
      const float nh[3] = {a.normal[px], a.normal[HW + px], a.normal[2 * HW + px]};
      if (a.tnormal && nN > 0) {
        const float t[3] = {a.tnormal[px], a.tnormal[HW + px], a.tnormal[2 * HW + px]};
        if (t[0] * t[0] + t[1] * t[1] + t[2] * t[2] > 0.f) {
          lng = 1.0 - (double)(nh[0] * t[0] + nh[1] * t[1] + nh[2] * t[2]);
          const float cf = a.lambda_n * a.lambda_ng / (float)nN;
          gn[0] -= cf * t[0]; gn[1] -= cf * t[1]; gn[2] -= cf * t[2];
        }
      }
      if (inner) {
        if (mE & mW & mU & mD) {
          float de[3], dw[3], du[3], dd[3];
          beam_dir(a, j, ip, de); beam_dir(a, j, im, dw); beam_dir(a, j - 1, i, du); beam_dir(a, j + 1, i, dd);
          const float dp[3] = {re * de[0] - rw * dw[0], re * de[1] - rw * dw[1], re * de[2] - rw * dw[2]};
          const float dt[3] = {ru * du[0] - rd * dd[0], ru * du[1] - rd * dd[1], ru * du[2] - rd * dd[2]};
          const float m[3] = {dp[1] * dt[2] - dp[2] * dt[1], dp[2] * dt[0] - dp[0] * dt[2], dp[0] * dt[1] - dp[1] * dt[0]};
          const float mn = sqrtf(m[0] * m[0] + m[1] * m[1] + m[2] * m[2]);
          if (mn >= 1e-12f) {
            ns_cnt = 1;
            const float im_ = 1.f / mn;
            const float mh[3] = {m[0] * im_, m[1] * im_, m[2] * im_};
            const float pr = mh[0] * nh[0] + mh[1] * nh[1] + mh[2] * nh[2];
            lns = 1.0 + (double)pr;                        // 1 - N^.N^s with N^s = -m^
            const float cf = a.lambda_n * a.lambda_ns * invM;
            gn[0] += cf * mh[0]; gn[1] += cf * mh[1]; gn[2] += cf * mh[2];
            if (!a.detach && cf != 0.f) {
              const float gm[3] = {cf * (nh[0] - pr * mh[0]) * im_, cf * (nh[1] - pr * mh[1]) * im_, cf * (nh[2] - pr * mh[2]) * im_};
              const float Gp[3] = {dt[1] * gm[2] - dt[2] * gm[1], dt[2] * gm[0] - dt[0] * gm[2], dt[0] * gm[1] - dt[1] * gm[0]};
              const float Gt[3] = {gm[1] * dp[2] - gm[2] * dp[1], gm[2] * dp[0] - gm[0] * dp[2], gm[0] * dp[1] - gm[1] * dp[0]};
              atomicAdd(&a.gD[pe], de[0] * Gp[0] + de[1] * Gp[1] + de[2] * Gp[2]);
              atomicAdd(&a.gD[pw], -(dw[0] * Gp[0] + dw[1] * Gp[1] + dw[2] * Gp[2]));
              atomicAdd(&a.gD[pu], du[0] * Gt[0] + du[1] * Gt[1] + du[2] * Gt[2]);
              atomicAdd(&a.gD[pd], -(dd[0] * Gt[0] + dd[1] * Gt[1] + dd[2] * Gt[2]));
            }
          }
        }
      }
    }
    a.gN[px] = gn[0]; a.gN[HW + px] = gn[1]; a.gN[2 * HW + px] = gn[2];
  } else if (px < HW) {
    a.gN[px] = 0.f; a.gN[HW + px] = 0.f; a.gN[2 * HW + px] = 0.f;
  }
  // block reduction of the three sums, one atomic each; the last block writes the scalars
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    ld += __shfl_xor_sync(0xffffffffu, ld, o);
    lng += __shfl_xor_sync(0xffffffffu, lng, o);
    lns += __shfl_xor_sync(0xffffffffu, lns, o);
    la += __shfl_xor_sync(0xffffffffu, la, o);
    ns_cnt += __shfl_xor_sync(0xffffffffu, ns_cnt, o);
  }
  if (lane == 0) { s_red[0][warp] = ld; s_red[1][warp] = lng; s_red[2][warp] = lns; s_red[3][warp] = la; s_cnt[warp] = ns_cnt; }
  __syncthreads();
  if (threadIdx.x == 0) {
    double t0 = 0, t1 = 0, t2 = 0, t3 = 0;
    unsigned int c = 0;
    for (int w = 0; w < 8; ++w) { t0 += s_red[0][w]; t1 += s_red[1][w]; t2 += s_red[2][w]; t3 += s_red[3][w]; c += s_cnt[w]; }
    if (t3 != 0.0) atomicAdd(&a.ws->La, t3);
    if (t0 != 0.0) atomicAdd(&a.ws->Ld, t0);
    if (t1 != 0.0) atomicAdd(&a.ws->Lng, t1);
    if (t2 != 0.0) atomicAdd(&a.ws->Lns, t2);
    if (c) atomicAdd(&a.ws->nS, c);
    __threadfence();
    if (atomicAdd(&a.ws->done, 1u) == gridDim.x - 1) {
      __threadfence();
      const volatile LossWs* w = a.ws;
      const double Ld = nM ? w->Ld / (double)nM : 0.0;
      const double Lng = nN ? w->Lng / (double)nN : 0.0;
      const double Lns = nM ? w->Lns / (double)nM : 0.0;
      const double La = nM ? w->La / (double)nM : 0.0;
      a.loss[1] = (float)Ld; a.loss[2] = (float)Lng; a.loss[3] = (float)Lns;
      if (a.n_loss > 4) a.loss[4] = (float)La;
      a.loss[0] = (float)(Ld + (double)a.lambda_alpha * La +
                          (double)a.lambda_n * ((double)a.lambda_ng * Lng + (double)a.lambda_ns * Lns));
    }
  }
}

}  // namespace

cudaError_t launch_loss(const SensorDev& sd, const float* range, const float* alpha, const float* normal,
                        const float* target_range, const float* target_normal, const uint8_t* keep_mask,
                        float lambda_alpha, float alpha_eps, int n_loss, float lambda_n, float lambda_ng,
                        float lambda_ns, int detach_surf, char* lws, float* loss, float* gD, float* gA, float* gN,
                        cudaStream_t st) {
  LossArgs a;
  a.alpha = alpha; a.lambda_alpha = lambda_alpha; a.alpha_eps = alpha_eps; a.n_loss = n_loss;
  a.H = sd.H; a.W = sd.W; a.elev_max = sd.elev_max; a.dphi = sd.dphi; a.dth = sd.dth;
  a.range = range; a.normal = normal; a.target = target_range; a.tnormal = target_normal; a.keep = keep_mask;
  a.lambda_n = lambda_n; a.lambda_ng = lambda_ng; a.lambda_ns = lambda_ns; a.detach = detach_surf;
  a.ws = reinterpret_cast<LossWs*>(lws);
  a.beams = reinterpret_cast<double*>(lws + kLossHdr);
  a.blk_cnt = reinterpret_cast<uint2*>(lws + kLossHdr + (size_t)(2 * sd.W + 2 * sd.H) * sizeof(double));
  a.loss = loss; a.gD = gD; a.gA = gA; a.gN = gN;
  const size_t HW = (size_t)sd.H * sd.W;
  const unsigned int grid = (unsigned int)((HW + 255) / 256);
  cudaError_t e = launch_pdl(loss_count_kernel, dim3(grid), dim3(256), 0, st, a);
  if (e != cudaSuccess) return e;
  loss_grad_kernel<<<grid, 256, 0, st>>>(a);
  return cudaGetLastError();
}

}  // namespace lgs
