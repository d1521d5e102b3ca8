// Internal declarations shared by the CUDA translation units of liblgs.so.
// (Nothing here is shared with oracle/: the oracle has its own definitions.)
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stddef.h>
#include "../../include/lgs.h"

namespace lgs {

constexpr int kTileW = LGS_TILE_W, kTileH = LGS_TILE_H;   // 8 x 4 pixel list tiles: one pixel per lane of a warp
static_assert(kTileW * kTileH == 32, "one pixel per lane");
constexpr int kIdBits = 24;              // surfel index bits of a sorted value (N <= 2^24)
constexpr int kProjThreads = 128;        // K1a / K1c: one surfel per thread
constexpr int kTileStride = 32;          // words between the atomic counters of consecutive tiles (one 128 B line each)
constexpr int kSortBigBucket = 11;       // K3: lists in length bucket >= 11 (n >= 1024) go to the big-class kernel
constexpr int kRadixBits = 8;
constexpr int kRadix = 1 << kRadixBits;
constexpr int kRecVec = 6;               // per-surfel record: 6 x float4 (96 B; the forward reads 5)
constexpr int kRecFloats = 4 * kRecVec;
constexpr int kPartFloats = 16;          // per-surfel gradient partial sums (13 used), one 64 B row

// cut-offs (reading R4 / R15)
#define LGS_ALPHA_MIN (1.0f / 255.0f)
#define LGS_ALPHA_MAX 0.99f
#define LGS_RHO2_MAX 9.0f
#define LGS_T_MIN 1e-4f
#define LGS_DEN_MIN 1e-6f

// Device-resident counters; zeroed at the start of every forward.
struct Header {
  unsigned int n_tasks;           // backward work items listed by the forward
  unsigned int n_visible;         // surfels with a non-empty rect
  unsigned int overflow;          // 1 if n_keys_total > max_keys
  unsigned int n_keys;            // keys actually present (= total, or 0 on overflow)
  unsigned long long n_keys_total;  // keys the frame needs
  unsigned long long n_contrib;   // contributing (pixel, surfel) pairs of the last forward
  unsigned int n_big;             // tiles with >= 2^(kSortBigBucket-1) keys: the first n_big entries of the schedule
  unsigned int n_tuples;          // (surfel, tile) tuples appended by the projection (= n_keys_total)
  unsigned int pad[6];
};
static_assert(sizeof(Header) <= 256, "header must fit its slot");

constexpr int kMaxFrames = LGS_MAX_FRAMES;   // keyframes of one batched call (frame id folded into the tile id)

// Sensor constants precomputed on the host in fp64 (same IEEE expressions as DESIGN.md's rule).  A batched call
// (lgs_render_*_batch) renders F keyframes that share the grid and differ in pose: tile ids
// run over F * ntiles_f tiles (frame f owns [f ntiles_f, (f+1) ntiles_f)), per-(frame, surfel) arrays are indexed
// f * N + i.  F = 1 is the single-frame call.
struct SensorDev {
  int H, W, ntc, ntr;
  int ntiles_f;     // tiles of one frame
  int ntiles;       // F * ntiles_f
  int F;
  long long N;      // surfels of the map (frame stride of the per-(frame, surfel) arrays)
  float r_min, r_max;
  double elev_max, dphi, dth;
  float cos_emax, sin_emax, cos_emin, sin_emin;   // (the projection's fp32 pre-cull)
};
// The poses of the frames (only the projection and the chain rule need them): row-major R_ws and t_ws.
struct PoseSet {
  double R[kMaxFrames][9];
  double t[kMaxFrames][3];
};

// Workspace carve-up (byte offsets), identical for forward / backward / query.
struct Layout {
  size_t hdr, tile_ctr, zero_end;     // tile_ctr: per tile one 128 B line {key count, ...}
  size_t tile_ranges, tile_order, beams, emit, rec, bhdr, part, keys0, keys1, vals0, vals1, pix, sums, pmask, tasks, pixgeo, anchor, total;
  size_t nslots;  // (tile, chunk) summary slots
  int n_proj_cta, proj_batch;
  int64_t cap;  // max_keys (>= 1)
};

// (range_gated only chooses the projection's grid shape; the byte offsets do not depend on it)
Layout make_layout(int64_t N, int H, int W, int64_t max_keys, int F = 1, bool range_gated = false);
SensorDev make_sensor(const lgs_sensor& s, int64_t N = 0, int F = 1);
PoseSet make_poses(const lgs_sensor* s, int F);

// ---- launchers (each enqueues on `st`, returns cudaGetLastError()) -------------
cudaError_t launch_project(const lgs_gaussians& g, const SensorDev& sd, const PoseSet& poses, const Layout& L, char* ws,
                           cudaStream_t st);
cudaError_t launch_ranges(const SensorDev& sd, const Layout& L, char* ws, cudaStream_t st);
cudaError_t launch_emit(const lgs_gaussians& g, const SensorDev& sd, const Layout& L, char* ws, cudaStream_t st);
// Sorts every segment [ranges[2t], ranges[2t+1]) of (keys0, vals0) by (key, value); tmp buffers
// are used only by the longest segments.  kv != NULL: the unsorted input of segment t is the interleaved
// (key, value) pairs kv[ranges[2t] ...) instead; the sorted output still goes to (keys0, vals0).  `sched` (may be NULL: every segment of `ranges` in order) = segment
// schedule {segment, start, end, -}, longest first, with *n_big (may be NULL) the number of leading big-class
// segments in it.
cudaError_t launch_tile_sort(uint32_t* keys0, uint32_t* keys1, uint32_t* vals0, uint32_t* vals1, const uint2* kv,
                             const unsigned int* ranges, const uint4* sched, const unsigned int* n_big, int nseg,
                             cudaStream_t st);
cudaError_t launch_composite_fwd(const SensorDev& sd, const Layout& L, char* ws, const uint32_t* vals,
                                 float* out_range, float* out_alpha, float* out_normal, cudaStream_t st);
cudaError_t launch_composite_bwd(const SensorDev& sd, const Layout& L, char* ws, const uint32_t* vals,
                                 const float* gD, const float* gA, const float* gN, cudaStream_t st);
// Zeroes the backward's counters and the per-surfel partial sums (launched with programmatic stream serialisation:
// nothing that precedes a backward in a stream reads or writes them, so it runs beside the preceding kernel).
cudaError_t launch_clear_partials(const SensorDev& sd, const Layout& L, char* ws, cudaStream_t st);
cudaError_t launch_chain(const lgs_gaussians& g, const SensorDev& sd, const PoseSet& poses, const Layout& L, char* ws, float* g_mean,
                         float* g_quat, float* g_scale, float* g_opacity, int accumulate, cudaStream_t st);
cudaError_t launch_loss(const SensorDev& sd, const float* range, const float* alpha, const float* normal,
                        const float* target_range, const float* target_normal, const uint8_t* keep_mask,
                        float lambda_alpha, float alpha_eps, int n_loss, float lambda_n, float lambda_ng,
                        float lambda_ns, int detach_surf, char* lws, float* loss, float* gD, float* gA, float* gN,
                        cudaStream_t st);
cudaError_t launch_scan(const SensorDev& sd, const float* points, const float* normals, int64_t M, void* zbuf,
                        float* out_range, float* out_normal, cudaStream_t st);
size_t prune_workspace_bytes(int64_t N);
// keep != NULL: compaction by keep flags (lgs_compact); else keep iff opacity >= alpha_min (lgs_prune_compact)
cudaError_t launch_prune(int64_t N, float alpha_min, const unsigned char* keep, const float* const in[7],
                         float* const out[7], long long* n_out, void* workspace, cudaStream_t st);
// map management (lgs_manage.cu)
size_t manage_workspace_bytes(int64_t N);
size_t cover_workspace_bytes(int64_t N, int64_t ncells);
cudaError_t launch_control_score(int64_t N, const float* sigma, const float* res, const float* bounds, const float* w,
                                 float eps, float* c, cudaStream_t st);
cudaError_t launch_quantile(int64_t N, const float* x, long long krank, float* out, void* workspace, cudaStream_t st);
cudaError_t launch_split(int64_t N, const float* c, const float* thr, float alpha_min, unsigned int cap, float shift,
                         float shrink, float* mean, float* quat, float* log_scale, float* opacity, float* scale, float* m,
                         float* v, unsigned char* flags_out, long long* n_new, void* workspace, cudaStream_t st);
struct CoverParams {
  int axis_a, axis_b;            // world axes of the projection plane
  float origin_a, origin_b, cell;
  int dim_a, dim_b;
  float alpha_min, kappa, q_cover, s_max;
  unsigned int cap;
};
cudaError_t launch_cover_prune(int64_t N, const float* mean, const float* quat, float* scale, float* log_scale,
                               const float* opacity, const float* c, const float* thr, const CoverParams& P,
                               unsigned char* keep, long long* n_removed, void* workspace, cudaStream_t st);
cudaError_t launch_adam(int64_t N, float* mean, float* quat, float* log_scale, float* opacity, float* scale,
                        const float* g_mean, const float* g_quat, const float* g_scale, const float* g_opacity,
                        float* m, float* v, const lgs_adam& h, float* loss_scale, cudaStream_t st);
cudaError_t launch_unpack_lists(const SensorDev& sd, const Layout& L, const char* ws, int64_t N, uint64_t* keys_out,
                                uint32_t* vals_out, int32_t* rects_out, cudaStream_t st);

inline size_t align_up(size_t x, size_t a = 256) { return (x + a - 1) / a * a; }

// Number of SMs of the current device (cached per device; 148 on a B200).
int sm_count();

// Programmatic dependent launch (cudaLaunchAttributeProgrammaticStreamSerialization): the grid may become resident
// while its predecessor in the stream still runs.  RULE: a kernel launched this way executes
// griddepcontrol.wait on every path before it retires -- at its top if it reads its predecessor's output, as its
// last statement otherwise -- so that "this grid has completed" implies "everything before it has completed" for
// whatever the stream runs next.  lgs_debug_set_pdl(0) turns the attribute off (plain stream order; tests).
bool pdl_enabled();
template <typename... KArgs, typename... Args>
inline cudaError_t launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st,
                              Args&&... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = pdl_enabled() ? 1 : 0;
  cfg.attrs = attr; cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, kernel, static_cast<KArgs>(args)...);
}

// Per-kernel CUDA-event timing (lgs_profile_*): RAII bracket around a launch group.
void prof_mark(int slot, bool end, cudaStream_t st);
struct ProfScope {
  int slot; cudaStream_t st;
  ProfScope(int s, cudaStream_t stream) : slot(s), st(stream) { prof_mark(slot, false, st); }
  ~ProfScope() { prof_mark(slot, true, st); }
};

}  // namespace lgs
