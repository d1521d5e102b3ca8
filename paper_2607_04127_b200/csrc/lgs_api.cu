// extern "C" entry points of liblgs.so (include/lgs.h): argument validation, workspace
// carve-up and kernel sequencing.  No allocation, no synchronisation (except lgs_query /
// lgs_debug_*), everything enqueued on the caller's stream.
#include <cmath>
#include <cstring>
#include "lgs_internal.cuh"

namespace lgs {

Layout make_layout(int64_t N, int H, int W, int64_t max_keys, int F, bool range_gated) {
  Layout L;
  std::memset(&L, 0, sizeof(L));
  const int ntc = (W + kTileW - 1) / kTileW, ntr = (H + kTileH - 1) / kTileH;
  const size_t ntiles_f = (size_t)ntc * ntr;
  const size_t nf = (size_t)(F > 0 ? F : 1);
  const size_t ntiles = ntiles_f * nf;                 // frame id folded into the tile id
  const size_t Nn = (size_t)(N > 0 ? N : 1) * nf;      // per-(frame, surfel) rows
  L.cap = max_keys > 0 ? max_keys : 1;
  // Pairs per thread of the projection.  With a finite r_max (a map larger than the sensor's reach: the pre-cull of the
  // projection then removes most pairs) a CTA takes up to 8 pairs per thread, so that the survivors fill whole warps --
  // once the grid exceeds ~2 waves of a B200 (148 SMs x 1,024 threads); otherwise 1 (measured: without a range gate the
  // pre-cull removes < 20 % of the pairs and the longer CTAs cost more than the packing saves).
  L.proj_batch = range_gated ? (int)(Nn / (2 * 148 * 1024)) : 1;
  L.proj_batch = L.proj_batch < 1 ? 1 : (L.proj_batch > 8 ? 8 : L.proj_batch);
  L.n_proj_cta = (int)((Nn + (size_t)L.proj_batch * kProjThreads - 1) / ((size_t)L.proj_batch * kProjThreads));
  size_t o = 0;
  L.hdr = o; o += align_up(sizeof(Header));
  L.tile_ctr = o; o += align_up(ntiles * kTileStride * 4);
  L.zero_end = o;
  L.tile_ranges = o; o += align_up(ntiles * 8);
  L.tile_order = o; o += align_up(ntiles * 16);   // schedule entries {tile, start, end, -}
  L.beams = o; o += align_up((size_t)(2 * W + 2 * H) * 8);
  L.emit = o; o += align_up(Nn * 16);
  L.rec = o; o += align_up(Nn * kRecFloats * 4);
  L.bhdr = o; o += 256;                     // backward counters
  L.part = o; o += align_up(Nn * kPartFloats * 4);
  L.keys0 = o; o += align_up((size_t)L.cap * 4);
  L.keys1 = o; o += align_up((size_t)L.cap * 4);
  L.vals0 = o; o += align_up((size_t)L.cap * 4);
  L.vals1 = o; o += align_up((size_t)L.cap * 4);
  L.pix = o; o += align_up((size_t)H * W * nf * 8);
  L.nslots = (size_t)L.cap / 32 + ntiles + 1;
  L.sums = o; o += align_up(L.nslots * 6 * 32 * 4);
  L.pmask = o; o += align_up(L.nslots * 32 * 4);
  L.tasks = o; o += align_up((L.nslots + ntiles + 1) * 16);     // at most one per chunk
  L.pixgeo = o; o += align_up((size_t)H * W * 16);              // (the frames share the grid)
  L.anchor = o; o += align_up(ntiles_f * 32);
  L.total = o;
  return L;
}

SensorDev make_sensor(const lgs_sensor& s, int64_t N, int F) {
  SensorDev d;
  d.H = s.H; d.W = s.W;
  d.ntc = (s.W + kTileW - 1) / kTileW; d.ntr = (s.H + kTileH - 1) / kTileH;
  d.ntiles_f = d.ntc * d.ntr;
  d.F = F > 0 ? F : 1;
  d.ntiles = d.ntiles_f * d.F;
  d.N = N;
  d.r_min = s.r_min; d.r_max = s.r_max;
  d.elev_max = (double)s.elev_max;
  d.dphi = (2.0 * 3.14159265358979323846) / (double)s.W;
  d.dth = ((double)s.elev_max - (double)s.elev_min) / (double)s.H;
  d.cos_emax = (float)std::cos((double)s.elev_max); d.sin_emax = (float)std::sin((double)s.elev_max);
  d.cos_emin = (float)std::cos((double)s.elev_min); d.sin_emin = (float)std::sin((double)s.elev_min);
  return d;
}

PoseSet make_poses(const lgs_sensor* s, int F) {
  PoseSet p;
  std::memset(&p, 0, sizeof(p));
  for (int f = 0; f < F && f < kMaxFrames; ++f) {
    for (int r = 0; r < 3; ++r) {
      for (int c = 0; c < 3; ++c) p.R[f][3 * r + c] = (double)s[f].T_ws[4 * r + c];
      p.t[f][r] = (double)s[f].T_ws[4 * r + 3];
    }
  }
  return p;
}

// Per-device facts (compute capability, SM count), looked up once per device: a process may drive several GPUs.
namespace {
constexpr int kMaxDevices = 64;
struct DeviceInfo { int state = 0; int major = 0; int sms = 0; };     // state: 0 unknown, 1 known
DeviceInfo g_dev[kMaxDevices];
const DeviceInfo* device_info() {
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) return nullptr;
  DeviceInfo& d = g_dev[dev];
  if (d.state == 0) {                 // (benign race: every thread writes the same values)
    int major = 0, sms = 0;
    if (cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess) return nullptr;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return nullptr;
    d.major = major; d.sms = sms; d.state = 1;
  }
  return &d;
}
bool g_pdl = true;
}  // namespace

static bool device_ok() {
  const DeviceInfo* d = device_info();
  return d && d->major == 10;
}

int sm_count() {
  const DeviceInfo* d = device_info();
  return (d && d->sms > 0) ? d->sms : 148;
}

bool pdl_enabled() { return g_pdl; }

// ---- lgs_profile_*: CUDA events around launch groups ------------------------------------------
static struct {
  bool on = false, created = false;
  cudaEvent_t ev[2 * LGS_PROF_SLOTS];
  bool used[LGS_PROF_SLOTS] = {false};
} g_prof;

void prof_mark(int slot, bool end, cudaStream_t st) {
  if (!g_prof.on || !g_prof.created) return;
  cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
  if (cudaStreamIsCapturing(st, &cs) != cudaSuccess || cs != cudaStreamCaptureStatusNone) return;
  cudaEventRecord(g_prof.ev[2 * slot + (end ? 1 : 0)], st);
  if (end) g_prof.used[slot] = true;
}

// The kernels read / write rows through 16-byte (float4) and 8-byte (float2) vector accesses: every array base
// pointer must be 16-byte aligned (NULL passes: optional arrays).
static bool al16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }
template <typename... P>
static bool all_al16(P... p) { return (al16(p) && ...); }

static bool sensor_ok(const lgs_sensor* s) {
  if (!s) return false;
  if (s->H < 1 || s->W < 1 || s->H > 32767 || s->W > 32767) return false;
  if (!(s->elev_min < s->elev_max)) return false;
  if (!(s->r_min >= 0.f) || !(s->r_max >= s->r_min)) return false;
  for (int k = 0; k < 12; ++k) if (!std::isfinite(s->T_ws[k])) return false;
  return true;
}

}  // namespace lgs

using namespace lgs;

extern "C" {

const char* lgs_version(void) { return "lgs 0.1 (sm_100a)"; }

size_t lgs_workspace_bytes(int64_t N, int32_t H, int32_t W, int64_t max_keys) {
  if (N < 0 || H < 1 || W < 1 || H > 32767 || W > 32767 || max_keys < 0 || max_keys >= (1ll << 30) || N > (1ll << kIdBits)) return 0;
  return make_layout(N, H, W, max_keys).total;
}

static bool frames_ok(const lgs_sensor* s, int32_t F) {
  if (!s || F < 1 || F > kMaxFrames) return false;
  for (int f = 0; f < F; ++f) {
    if (!sensor_ok(s + f)) return false;
    if (s[f].H != s[0].H || s[f].W != s[0].W || s[f].elev_min != s[0].elev_min || s[f].elev_max != s[0].elev_max ||
        s[f].r_min != s[0].r_min || !(s[f].r_max == s[0].r_max))
      return false;
  }
  return true;
}

size_t lgs_workspace_bytes_batch(int64_t N, int32_t H, int32_t W, int64_t max_keys, int32_t F) {
  if (F < 1 || F > kMaxFrames) return 0;
  if (N < 0 || H < 1 || W < 1 || H > 32767 || W > 32767 || max_keys < 0 || max_keys >= (1ll << 30) || N > (1ll << kIdBits)) return 0;
  return make_layout(N, H, W, max_keys, F).total;
}

lgs_status lgs_render_forward_batch(const lgs_gaussians* g, const lgs_sensor* s, int32_t F, void* workspace,
                                    size_t workspace_bytes, int64_t max_keys, float* out_range, float* out_alpha,
                                    float* out_normal, lgs_stream stream) {
  if (!g || !frames_ok(s, F) || !workspace || !out_range || !out_alpha) return LGS_ERR_INVALID_ARG;
  if (g->N < 0 || g->N > (1ll << kIdBits) || max_keys < 0 || max_keys >= (1ll << 30)) return LGS_ERR_INVALID_ARG;
  if (g->N > 0 && (!g->mean || !g->quat || !g->scale || !g->opacity)) return LGS_ERR_INVALID_ARG;
  if (!all_al16(g->mean, g->quat, g->scale, g->opacity, out_range, out_alpha, out_normal)) return LGS_ERR_INVALID_ARG;
  if ((reinterpret_cast<uintptr_t>(workspace) & 255u) != 0) return LGS_ERR_INVALID_ARG;
  if (!device_ok()) return LGS_ERR_UNSUPPORTED_DEVICE;
  const Layout L = make_layout(g->N, s->H, s->W, max_keys, F, std::isfinite(s->r_max));
  if (workspace_bytes < L.total) return LGS_ERR_WORKSPACE_TOO_SMALL;
  const SensorDev sd = make_sensor(*s, g->N, F);
  const PoseSet poses = make_poses(s, F);
  char* ws = static_cast<char*>(workspace);
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  {
    ProfScope ps(LGS_PROF_PROJECT, st);
    if (cudaMemsetAsync(ws, 0, L.zero_end, st) != cudaSuccess) return LGS_ERR_CUDA;
    if (launch_project(*g, sd, poses, L, ws, st) != cudaSuccess) return LGS_ERR_CUDA;
  }
  {
    ProfScope ps(LGS_PROF_EMIT, st);
    if (launch_ranges(sd, L, ws, st) != cudaSuccess) return LGS_ERR_CUDA;
    if (launch_emit(*g, sd, L, ws, st) != cudaSuccess) return LGS_ERR_CUDA;
  }
  uint32_t* vals = reinterpret_cast<uint32_t*>(ws + L.vals0);
  {
    ProfScope ps(LGS_PROF_SORT, st);
    if (launch_tile_sort(reinterpret_cast<uint32_t*>(ws + L.keys0), reinterpret_cast<uint32_t*>(ws + L.keys1), vals,
                         reinterpret_cast<uint32_t*>(ws + L.vals1),
                         reinterpret_cast<const uint2*>(ws + L.sums + (size_t)L.cap * 16),     // placement's output
                         reinterpret_cast<const unsigned int*>(ws + L.tile_ranges),
                         reinterpret_cast<const uint4*>(ws + L.tile_order),
                         &reinterpret_cast<const Header*>(ws + L.hdr)->n_big, sd.ntiles, st) != cudaSuccess)
      return LGS_ERR_CUDA;
  }
  {
    ProfScope ps(LGS_PROF_COMPOSITE_FWD, st);
    if (launch_composite_fwd(sd, L, ws, vals, out_range, out_alpha, out_normal, st) != cudaSuccess)
      return LGS_ERR_CUDA;
  }
  return LGS_OK;
}

lgs_status lgs_render_forward(const lgs_gaussians* g, const lgs_sensor* s, void* workspace, size_t workspace_bytes,
                              int64_t max_keys, float* out_range, float* out_alpha, float* out_normal,
                              lgs_stream stream) {
  return lgs_render_forward_batch(g, s, 1, workspace, workspace_bytes, max_keys, out_range, out_alpha, out_normal, stream);
}

lgs_status lgs_render_backward_batch(const lgs_gaussians* g, const lgs_sensor* s, int32_t F, void* workspace,
                                     size_t workspace_bytes, int64_t max_keys, const float* dL_drange,
                                     const float* dL_dalpha, const float* dL_dnormal, float* g_mean, float* g_quat,
                                     float* g_scale, float* g_opacity, int accumulate, lgs_stream stream) {
  if (!g || !frames_ok(s, F) || !workspace || !dL_drange) return LGS_ERR_INVALID_ARG;
  if (g->N < 0 || g->N > (1ll << kIdBits) || max_keys < 0 || max_keys >= (1ll << 30)) return LGS_ERR_INVALID_ARG;
  if (g->N > 0 && (!g->mean || !g->quat || !g->scale || !g->opacity || !g_mean || !g_quat || !g_scale || !g_opacity))
    return LGS_ERR_INVALID_ARG;
  if (!all_al16(g->mean, g->quat, g->scale, g->opacity, dL_drange, dL_dalpha, dL_dnormal, g_mean, g_quat, g_scale,
                g_opacity))
    return LGS_ERR_INVALID_ARG;
  if ((reinterpret_cast<uintptr_t>(workspace) & 255u) != 0) return LGS_ERR_INVALID_ARG;
  if (!device_ok()) return LGS_ERR_UNSUPPORTED_DEVICE;
  const Layout L = make_layout(g->N, s->H, s->W, max_keys, F);
  if (workspace_bytes < L.total) return LGS_ERR_WORKSPACE_TOO_SMALL;
  const SensorDev sd = make_sensor(*s, g->N, F);
  const PoseSet poses = make_poses(s, F);
  char* ws = static_cast<char*>(workspace);
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  const uint32_t* vals = reinterpret_cast<uint32_t*>(ws + L.vals0);
  {
    ProfScope ps(LGS_PROF_COMPOSITE_BWD, st);
    if (launch_clear_partials(sd, L, ws, st) != cudaSuccess) return LGS_ERR_CUDA;
    if (launch_composite_bwd(sd, L, ws, vals, dL_drange, dL_dalpha, dL_dnormal, st) != cudaSuccess) return LGS_ERR_CUDA;
  }
  {
    ProfScope ps(LGS_PROF_CHAIN, st);
    if (launch_chain(*g, sd, poses, L, ws, g_mean, g_quat, g_scale, g_opacity, accumulate, st) != cudaSuccess)
      return LGS_ERR_CUDA;
  }
  return LGS_OK;
}

lgs_status lgs_render_backward(const lgs_gaussians* g, const lgs_sensor* s, void* workspace, size_t workspace_bytes,
                               int64_t max_keys, const float* dL_drange, const float* dL_dalpha,
                               const float* dL_dnormal, float* g_mean, float* g_quat, float* g_scale,
                               float* g_opacity, int accumulate, lgs_stream stream) {
  return lgs_render_backward_batch(g, s, 1, workspace, workspace_bytes, max_keys, dL_drange, dL_dalpha, dL_dnormal,
                                   g_mean, g_quat, g_scale, g_opacity, accumulate, stream);
}

size_t lgs_loss_workspace_bytes(int32_t H, int32_t W) {
  if (H < 1 || W < 1) return 0;
  // counters + beam table + per-block pixel counts of the count kernel (256 pixels per block)
  return 256 + (size_t)(2 * W + 2 * H) * sizeof(double) + (((size_t)H * W + 255) / 256) * 8;
}

static lgs_status loss_call(const lgs_sensor* s, const float* range, const float* alpha, const float* normal,
                            const float* target_range, const float* target_normal, const uint8_t* keep_mask,
                            float lambda_alpha, float alpha_eps, int n_loss, float lambda_n, float lambda_ng,
                            float lambda_ns, int detach_surf, void* loss_workspace, size_t loss_workspace_bytes,
                            float* loss, float* dL_drange, float* dL_dalpha, float* dL_dnormal, lgs_stream stream) {
  if (!sensor_ok(s) || !range || !normal || !target_range || !loss_workspace || !loss || !dL_drange || !dL_dalpha ||
      !dL_dnormal)
    return LGS_ERR_INVALID_ARG;
  if (lambda_alpha != 0.f && (!alpha || !(alpha_eps >= 0.f))) return LGS_ERR_INVALID_ARG;
  if ((reinterpret_cast<uintptr_t>(loss_workspace) & 7u) != 0) return LGS_ERR_INVALID_ARG;
  if (loss_workspace_bytes < lgs_loss_workspace_bytes(s->H, s->W)) return LGS_ERR_WORKSPACE_TOO_SMALL;
  if (!device_ok()) return LGS_ERR_UNSUPPORTED_DEVICE;
  const SensorDev sd = make_sensor(*s);
  ProfScope ps(LGS_PROF_LOSS, reinterpret_cast<cudaStream_t>(stream));
  if (launch_loss(sd, range, alpha, normal, target_range, target_normal, keep_mask, lambda_alpha, alpha_eps, n_loss,
                  lambda_n, lambda_ng, lambda_ns, detach_surf, static_cast<char*>(loss_workspace), loss, dL_drange,
                  dL_dalpha, dL_dnormal, reinterpret_cast<cudaStream_t>(stream)) != cudaSuccess)
    return LGS_ERR_CUDA;
  return LGS_OK;
}

lgs_status lgs_loss_range_normal(const lgs_sensor* s, const float* range, const float* alpha, const float* normal,
                                 const float* target_range, const float* target_normal, const uint8_t* keep_mask,
                                 float lambda_n, float lambda_ng, float lambda_ns, int detach_surf,
                                 void* loss_workspace, size_t loss_workspace_bytes, float* loss, float* dL_drange,
                                 float* dL_dalpha, float* dL_dnormal, lgs_stream stream) {
  return loss_call(s, range, alpha, normal, target_range, target_normal, keep_mask, 0.f, 0.f, 4, lambda_n, lambda_ng,
                   lambda_ns, detach_surf, loss_workspace, loss_workspace_bytes, loss, dL_drange, dL_dalpha, dL_dnormal,
                   stream);
}

lgs_status lgs_loss_mapping(const lgs_sensor* s, const float* range, const float* alpha, const float* normal,
                            const float* target_range, const float* target_normal, const uint8_t* keep_mask,
                            float lambda_alpha, float alpha_eps, float lambda_n, float lambda_ng, float lambda_ns,
                            int detach_surf, void* loss_workspace, size_t loss_workspace_bytes, float* loss,
                            float* dL_drange, float* dL_dalpha, float* dL_dnormal, lgs_stream stream) {
  if (!alpha) return LGS_ERR_INVALID_ARG;
  return loss_call(s, range, alpha, normal, target_range, target_normal, keep_mask, lambda_alpha, alpha_eps, 5,
                   lambda_n, lambda_ng, lambda_ns, detach_surf, loss_workspace, loss_workspace_bytes, loss, dL_drange,
                   dL_dalpha, dL_dnormal, stream);
}

lgs_status lgs_adam_step(int64_t N, float* mean, float* quat, float* log_scale, float* opacity, float* scale,
                         const float* g_mean, const float* g_quat, const float* g_scale, const float* g_opacity,
                         float* m, float* v, const lgs_adam* h, float* loss_scale, lgs_stream stream) {
  if (N < 0 || !h || !loss_scale) return LGS_ERR_INVALID_ARG;
  if (N > 0 && (!mean || !quat || !log_scale || !opacity || !scale || !g_mean || !g_quat || !g_scale || !g_opacity ||
                !m || !v))
    return LGS_ERR_INVALID_ARG;
  if (!all_al16(mean, quat, log_scale, opacity, scale, g_mean, g_quat, g_scale, g_opacity, m, v)) return LGS_ERR_INVALID_ARG;
  if ((!h->step_device && h->step < 1) || !(h->beta1 >= 0.f && h->beta1 < 1.f) || !(h->beta2 >= 0.f && h->beta2 < 1.f) || !(h->eps >= 0.f) ||
      !(h->alpha_lo <= h->alpha_hi))
    return LGS_ERR_INVALID_ARG;
  if (!device_ok()) return LGS_ERR_UNSUPPORTED_DEVICE;
  ProfScope ps(LGS_PROF_ADAM, reinterpret_cast<cudaStream_t>(stream));
  if (launch_adam(N, mean, quat, log_scale, opacity, scale, g_mean, g_quat, g_scale, g_opacity, m, v, *h, loss_scale,
                  reinterpret_cast<cudaStream_t>(stream)) != cudaSuccess)
    return LGS_ERR_CUDA;
  return LGS_OK;
}

size_t lgs_prune_workspace_bytes(int64_t N) {
  if (N < 0 || N > (1ll << kIdBits)) return 0;
  return prune_workspace_bytes(N);
}

static lgs_status compact_call(int64_t N, float alpha_min, const uint8_t* keep, const float* mean, const float* quat,
                               const float* log_scale, const float* opacity, const float* scale, const float* m,
                               const float* v, float* out_mean, float* out_quat, float* out_log_scale, float* out_opacity,
                               float* out_scale, float* out_m, float* out_v, int64_t* n_out, void* workspace,
                               size_t workspace_bytes, lgs_stream stream) {
  if (N < 0 || N > (1ll << kIdBits) || !n_out || !workspace) return LGS_ERR_INVALID_ARG;
  if (N > 0 && (!mean || !quat || !log_scale || !opacity || !out_mean || !out_quat || !out_log_scale || !out_opacity))
    return LGS_ERR_INVALID_ARG;
  if ((scale == nullptr) != (out_scale == nullptr) || (m == nullptr) != (out_m == nullptr) ||
      (v == nullptr) != (out_v == nullptr))
    return LGS_ERR_INVALID_ARG;
  if ((reinterpret_cast<uintptr_t>(workspace) & 3u) != 0 || (reinterpret_cast<uintptr_t>(n_out) & 7u) != 0)
    return LGS_ERR_INVALID_ARG;
  if (!all_al16(mean, quat, log_scale, opacity, scale, m, v, out_mean, out_quat, out_log_scale, out_opacity, out_scale,
                out_m, out_v))
    return LGS_ERR_INVALID_ARG;
  {   // the outputs must not alias the inputs (the scatter reads rows other CTAs may already have overwritten)
    const void* ins[7] = {mean, quat, log_scale, opacity, scale, m, v};
    const void* outs[7] = {out_mean, out_quat, out_log_scale, out_opacity, out_scale, out_m, out_v};
    const size_t width[7] = {3, 4, 2, 1, 2, 10, 10};
    for (int a = 0; a < 7; ++a)
      for (int b = 0; b < 7; ++b) {
        if (!ins[a] || !outs[b] || N == 0) continue;
        const char* i0 = static_cast<const char*>(ins[a]); const char* o0 = static_cast<const char*>(outs[b]);
        if (i0 < o0 + (size_t)N * width[b] * 4 && o0 < i0 + (size_t)N * width[a] * 4) return LGS_ERR_INVALID_ARG;
      }
  }
  if (workspace_bytes < prune_workspace_bytes(N)) return LGS_ERR_WORKSPACE_TOO_SMALL;
  if (!device_ok()) return LGS_ERR_UNSUPPORTED_DEVICE;
  const float* in[7] = {mean, quat, log_scale, opacity, scale, m, v};
  float* out[7] = {out_mean, out_quat, out_log_scale, out_opacity, out_scale, out_m, out_v};
  if (launch_prune(N, alpha_min, keep, in, out, reinterpret_cast<long long*>(n_out), workspace,
                   reinterpret_cast<cudaStream_t>(stream)) != cudaSuccess)
    return LGS_ERR_CUDA;
  return LGS_OK;
}

lgs_status lgs_prune_compact(int64_t N, float alpha_min, const float* mean, const float* quat, const float* log_scale,
                             const float* opacity, const float* scale, const float* m, const float* v, float* out_mean,
                             float* out_quat, float* out_log_scale, float* out_opacity, float* out_scale, float* out_m,
                             float* out_v, int64_t* n_out, void* workspace, size_t workspace_bytes, lgs_stream stream) {
  return compact_call(N, alpha_min, nullptr, mean, quat, log_scale, opacity, scale, m, v, out_mean, out_quat, out_log_scale,
                      out_opacity, out_scale, out_m, out_v, n_out, workspace, workspace_bytes, stream);
}

lgs_status lgs_compact(int64_t N, const uint8_t* keep, const float* mean, const float* quat, const float* log_scale,
                       const float* opacity, const float* scale, const float* m, const float* v, float* out_mean,
                       float* out_quat, float* out_log_scale, float* out_opacity, float* out_scale, float* out_m,
                       float* out_v, int64_t* n_out, void* workspace, size_t workspace_bytes, lgs_stream stream) {
  if (N > 0 && !keep) return LGS_ERR_INVALID_ARG;
  static const uint8_t none = 0;
  return compact_call(N, 0.f, keep ? keep : &none, mean, quat, log_scale, opacity, scale, m, v,
                      out_mean, out_quat, out_log_scale, out_opacity, out_scale, out_m, out_v, n_out, workspace,
                      workspace_bytes, stream);
}

lgs_status lgs_control_score(int64_t N, const float* sigma, const float* res, const float* bounds, const float* weights,
                             float eps, float* c, lgs_stream stream) {
  if (N < 0 || !bounds || !weights || !(eps >= 0.f)) return LGS_ERR_INVALID_ARG;
  if (N > 0 && (!sigma || !res || !c)) return LGS_ERR_INVALID_ARG;
  for (int k = 0; k < 3; ++k) if (!(bounds[2 * k + 1] > bounds[2 * k])) return LGS_ERR_INVALID_ARG;
  if (!device_ok()) return LGS_ERR_UNSUPPORTED_DEVICE;
  if (launch_control_score(N, sigma, res, bounds, weights, eps, c, reinterpret_cast<cudaStream_t>(stream)) != cudaSuccess)
    return LGS_ERR_CUDA;
  return LGS_OK;
}

size_t lgs_manage_workspace_bytes(int64_t N) {
  if (N < 0 || N > (1ll << kIdBits)) return 0;
  return manage_workspace_bytes(N);
}

lgs_status lgs_quantile(int64_t N, const float* x, double q, float* out, void* workspace, size_t workspace_bytes,
                        lgs_stream stream) {
  if (N < 0 || N > (1ll << kIdBits) || !out || !workspace || !(q >= 0.0 && q <= 1.0) || (N > 0 && !x)) return LGS_ERR_INVALID_ARG;
  if ((reinterpret_cast<uintptr_t>(workspace) & 255u) != 0) return LGS_ERR_INVALID_ARG;
  if (workspace_bytes < manage_workspace_bytes(N)) return LGS_ERR_WORKSPACE_TOO_SMALL;
  if (!device_ok()) return LGS_ERR_UNSUPPORTED_DEVICE;
  long long k = (long long)std::ceil(q * (double)N);
  k = k < 1 ? 1 : (k > N ? N : k);
  if (launch_quantile(N, x, k, out, workspace, reinterpret_cast<cudaStream_t>(stream)) != cudaSuccess) return LGS_ERR_CUDA;
  return LGS_OK;
}

lgs_status lgs_split(int64_t N, const float* c, const float* thr, float alpha_min, int64_t max_splits, float shift,
                     float shrink, float* mean, float* quat, float* log_scale, float* opacity, float* scale, float* m,
                     float* v, uint8_t* flags_out, int64_t* n_new, void* workspace, size_t workspace_bytes,
                     lgs_stream stream) {
  if (N < 0 || max_splits < 0 || N + max_splits > (1ll << kIdBits) || !thr || !n_new || !workspace || !(shrink > 0.f))
    return LGS_ERR_INVALID_ARG;
  if (N > 0 && (!c || !mean || !quat || !log_scale || !opacity)) return LGS_ERR_INVALID_ARG;
  if (!all_al16(mean, quat, log_scale, opacity, scale, m, v) || (reinterpret_cast<uintptr_t>(workspace) & 255u) != 0 ||
      (reinterpret_cast<uintptr_t>(n_new) & 7u) != 0)
    return LGS_ERR_INVALID_ARG;
  if (workspace_bytes < manage_workspace_bytes(N)) return LGS_ERR_WORKSPACE_TOO_SMALL;
  if (!device_ok()) return LGS_ERR_UNSUPPORTED_DEVICE;
  if (launch_split(N, c, thr, alpha_min, (unsigned int)max_splits, shift, shrink, mean, quat, log_scale, opacity, scale, m,
                   v, flags_out, reinterpret_cast<long long*>(n_new), workspace, reinterpret_cast<cudaStream_t>(stream)) !=
      cudaSuccess)
    return LGS_ERR_CUDA;
  return LGS_OK;
}

size_t lgs_cover_workspace_bytes(int64_t N, int32_t dim_a, int32_t dim_b) {
  if (N < 0 || N > (1ll << kIdBits) || dim_a < 1 || dim_b < 1 || (int64_t)dim_a * dim_b > (1ll << 28)) return 0;
  return cover_workspace_bytes(N, (int64_t)dim_a * dim_b);
}

lgs_status lgs_cover_prune_pass(int64_t N, const float* mean, const float* quat, float* scale, float* log_scale,
                                const float* opacity, const float* c, const float* thr, const lgs_cover_params* p,
                                uint8_t* keep, int64_t* n_removed, void* workspace, size_t workspace_bytes,
                                lgs_stream stream) {
  if (N < 0 || N > (1ll << kIdBits) || !p || !thr || !n_removed || !workspace) return LGS_ERR_INVALID_ARG;
  if (N > 0 && (!mean || !quat || !scale || !opacity || !c || !keep)) return LGS_ERR_INVALID_ARG;
  if (p->axis_a < 0 || p->axis_a > 2 || p->axis_b < 0 || p->axis_b > 2 || p->axis_a == p->axis_b || !(p->cell > 0.f) ||
      p->dim_a < 1 || p->dim_b < 1 || (int64_t)p->dim_a * p->dim_b > (1ll << 28) || !(p->kappa > 0.f) ||
      !(p->q_cover >= 0.f && p->q_cover <= 1.f) || !(p->s_max > 0.f) || p->max_removed < 0)
    return LGS_ERR_INVALID_ARG;
  if (!all_al16(mean, quat, scale, log_scale, opacity, c) || (reinterpret_cast<uintptr_t>(workspace) & 255u) != 0 ||
      (reinterpret_cast<uintptr_t>(n_removed) & 7u) != 0)
    return LGS_ERR_INVALID_ARG;
  if (workspace_bytes < cover_workspace_bytes(N, (int64_t)p->dim_a * p->dim_b)) return LGS_ERR_WORKSPACE_TOO_SMALL;
  if (!device_ok()) return LGS_ERR_UNSUPPORTED_DEVICE;
  CoverParams P;
  P.axis_a = p->axis_a; P.axis_b = p->axis_b; P.origin_a = p->origin_a; P.origin_b = p->origin_b; P.cell = p->cell;
  P.dim_a = p->dim_a; P.dim_b = p->dim_b; P.alpha_min = p->alpha_min; P.kappa = p->kappa; P.q_cover = p->q_cover;
  P.s_max = p->s_max; P.cap = (unsigned int)(p->max_removed > 0xffffffffll ? 0xffffffffll : p->max_removed);
  if (launch_cover_prune(N, mean, quat, scale, log_scale, opacity, c, thr, P, keep, reinterpret_cast<long long*>(n_removed),
                         workspace, reinterpret_cast<cudaStream_t>(stream)) != cudaSuccess)
    return LGS_ERR_CUDA;
  return LGS_OK;
}

lgs_status lgs_scan_to_range_image(const float* points, const float* normals, int64_t M, const lgs_sensor* s,
                                   void* zbuf, size_t zbuf_bytes, float* out_range, float* out_normal,
                                   lgs_stream stream) {
  if (!sensor_ok(s) || M < 0 || M > 0xffffffffll || (M > 0 && !points) || !zbuf || !out_range) return LGS_ERR_INVALID_ARG;
  if ((reinterpret_cast<uintptr_t>(zbuf) & 7u) != 0) return LGS_ERR_INVALID_ARG;
  if (zbuf_bytes < (size_t)s->H * s->W * 8) return LGS_ERR_WORKSPACE_TOO_SMALL;
  if (!device_ok()) return LGS_ERR_UNSUPPORTED_DEVICE;
  const SensorDev sd = make_sensor(*s);
  if (launch_scan(sd, points, normals, M, zbuf, out_range, out_normal, reinterpret_cast<cudaStream_t>(stream)) !=
      cudaSuccess)
    return LGS_ERR_CUDA;
  return LGS_OK;
}

lgs_status lgs_query(const void* workspace, int64_t N, int32_t H, int32_t W, int64_t max_keys, int64_t* n_visible,
                     int64_t* n_keys, int64_t* n_contrib, lgs_stream stream) {
  if (!workspace || N < 0 || H < 1 || W < 1 || max_keys < 0) return LGS_ERR_INVALID_ARG;
  const Layout L = make_layout(N, H, W, max_keys);
  Header h;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  if (cudaMemcpyAsync(&h, static_cast<const char*>(workspace) + L.hdr, sizeof(Header), cudaMemcpyDeviceToHost, st) !=
      cudaSuccess)
    return LGS_ERR_CUDA;
  if (cudaStreamSynchronize(st) != cudaSuccess) return LGS_ERR_CUDA;
  if (n_visible) *n_visible = (int64_t)h.n_visible;
  if (n_keys) *n_keys = (int64_t)h.n_keys_total;
  if (n_contrib) *n_contrib = (int64_t)h.n_contrib;
  return h.overflow ? LGS_ERR_KEY_OVERFLOW : LGS_OK;
}

lgs_status lgs_debug_tile_lists_batch(const void* workspace, const lgs_sensor* s, int32_t F, int64_t N, int64_t max_keys,
                                      uint64_t* keys_out, uint32_t* vals_out, const uint32_t** tile_ranges,
                                      int32_t* rects_out, lgs_stream stream) {
  if (!workspace || !sensor_ok(s) || F < 1 || F > kMaxFrames || N < 0 || max_keys < 0) return LGS_ERR_INVALID_ARG;
  const Layout L = make_layout(N, s->H, s->W, max_keys, F);
  const SensorDev sd = make_sensor(*s, N, F);
  const char* ws = static_cast<const char*>(workspace);
  if (tile_ranges) *tile_ranges = reinterpret_cast<const uint32_t*>(ws + L.tile_ranges);
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  if (launch_unpack_lists(sd, L, ws, N * F, keys_out, vals_out, rects_out, st) != cudaSuccess) return LGS_ERR_CUDA;
  if (cudaStreamSynchronize(st) != cudaSuccess) return LGS_ERR_CUDA;
  return LGS_OK;
}

lgs_status lgs_debug_tile_lists(const void* workspace, const lgs_sensor* s, int64_t N, int64_t max_keys,
                                uint64_t* keys_out, uint32_t* vals_out, const uint32_t** tile_ranges,
                                int32_t* rects_out, lgs_stream stream) {
  return lgs_debug_tile_lists_batch(workspace, s, 1, N, max_keys, keys_out, vals_out, tile_ranges, rects_out, stream);
}

lgs_status lgs_debug_set_pdl(int enabled) {
  g_pdl = enabled != 0;
  return LGS_OK;
}

lgs_status lgs_profile_enable(int on) {
  if (on && !g_prof.created) {
    for (int k = 0; k < 2 * LGS_PROF_SLOTS; ++k)
      if (cudaEventCreate(&g_prof.ev[k]) != cudaSuccess) return LGS_ERR_CUDA;
    g_prof.created = true;
  }
  g_prof.on = on != 0;
  for (int k = 0; k < LGS_PROF_SLOTS; ++k) g_prof.used[k] = false;
  return LGS_OK;
}

lgs_status lgs_profile_read(float* ms, lgs_stream stream) {
  if (!ms) return LGS_ERR_INVALID_ARG;
  if (cudaStreamSynchronize(reinterpret_cast<cudaStream_t>(stream)) != cudaSuccess) return LGS_ERR_CUDA;
  for (int k = 0; k < LGS_PROF_SLOTS; ++k) {
    ms[k] = 0.f;
    if (g_prof.created && g_prof.used[k]) {
      if (cudaEventElapsedTime(&ms[k], g_prof.ev[2 * k], g_prof.ev[2 * k + 1]) != cudaSuccess) ms[k] = 0.f;
      g_prof.used[k] = false;
    }
  }
  return LGS_OK;
}

const char* lgs_profile_slot_name(int slot) {
  static const char* names[LGS_PROF_SLOTS] = {"project", "emit", "tile_sort", "composite_fwd",
                                              "loss", "composite_bwd", "chain", "adam"};
  return (slot >= 0 && slot < LGS_PROF_SLOTS) ? names[slot] : "";
}

lgs_status lgs_debug_segmented_sort(uint32_t* keys, uint32_t* vals, uint32_t* tmp_keys, uint32_t* tmp_vals,
                                    const uint32_t* seg_ranges, int32_t n_segments, lgs_stream stream) {
  if (n_segments < 0) return LGS_ERR_INVALID_ARG;
  if (n_segments > 0 && (!keys || !vals || !tmp_keys || !tmp_vals || !seg_ranges)) return LGS_ERR_INVALID_ARG;
  if (!device_ok()) return LGS_ERR_UNSUPPORTED_DEVICE;
  if (launch_tile_sort(keys, tmp_keys, vals, tmp_vals, nullptr, seg_ranges, nullptr, nullptr, n_segments,
                       reinterpret_cast<cudaStream_t>(stream)) != cudaSuccess)
    return LGS_ERR_CUDA;
  return LGS_OK;
}

}  // extern "C"
