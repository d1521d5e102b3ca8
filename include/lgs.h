/* =============================================================================
 * lgs.h -- C ABI of the B200-native differentiable spherical surfel rasteriser.
 *
 * What it computes (arxiv/paper_2607_04127): the hot path of the paper's mapping
 * stage -- "render the Gaussian map under the same spherical projection pi_s(.),
 * producing (D^, A^, N^) on a shared grid" (section 3.1) and
 * "optimizes the Gaussian parameters Theta = {mu, q, s~, alpha} by comparing them
 * against the observations" (section 3.4), with the masked L1 range
 * loss (Eq. 10 left) and the normal loss (Eq. 11).
 * The paper does not define the rasteriser; the exact definition implemented here
 * (beam grid, ray/plane intersection, cut-offs, ordering) is DESIGN.md "Readings".
 *
 * Conventions common to every entry point
 *  - Every data pointer is a DEVICE pointer unless the comment says "host".
 *    Structs (lgs_gaussians, lgs_sensor) are read from HOST memory at call time.
 *  - The caller owns every buffer.  The library never allocates, frees or
 *    synchronises (except lgs_query and lgs_debug_*), enqueues all work on the
 *    given stream, and is CUDA-Graph capturable.
 *  - Argument errors are returned synchronously as lgs_status; no C++ exception
 *    crosses the boundary.  Data-dependent overflow (more tile keys than
 *    max_keys) is recorded in the workspace: the frame then renders as all zeros,
 *    backward produces zero gradients, and lgs_query reports the count needed.
 *  - Layouts are row-major, fp32: images [H,W] (row 0 = elev_max, column 0 =
 *    azimuth -pi, full 2*pi), normal images [3,H,W], parameters [N,3] / [N,4] /
 *    [N,2] / [N].
 *  - Only sm_100 (B200) devices are supported: LGS_ERR_UNSUPPORTED_DEVICE
 *    otherwise.  There is no CPU fallback.
 * ============================================================================= */
#ifndef LGS_H_
#define LGS_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  LGS_OK = 0,
  LGS_ERR_INVALID_ARG = 1,
  LGS_ERR_WORKSPACE_TOO_SMALL = 2,
  LGS_ERR_KEY_OVERFLOW = 3,       /* reported by lgs_query only */
  LGS_ERR_CUDA = 4,
  LGS_ERR_UNSUPPORTED_DEVICE = 5,
  LGS_ERR_STATIC_LIMIT = 6        /* lgs_scan_to_range_image_static only: H * W > LGS_SCAN_STATIC_MAX_PIXELS */
} lgs_status;

/* Same type as cudaStream_t (CUstream_st*); NULL is the legacy default stream. */
typedef struct CUstream_st* lgs_stream;

/* The map: G = {(mu_i, q_i, s~_i, alpha_i)}.  Parameters are taken in
 * ACTIVATED space (metres, opacity in [0,1]); the chain rule to the paper's
 * log-scale belongs to the optimiser (reading R8). */
typedef struct {
  const float* mean;     /* [N,3] world frame */
  const float* quat;     /* [N,4] (w,x,y,z), Hamilton; need not be unit, normalised inside */
  const float* scale;    /* [N,2] in-plane standard deviations s0 (along R(q)e0), s1 (along R(q)e1) */
  const float* opacity;  /* [N] */
  int64_t N;             /* 0 <= N <= LGS_MAX_SURFELS */
} lgs_gaussians;

/* Largest map one call accepts (the sorted list values keep the surfel index in 24 bits). */
#define LGS_MAX_SURFELS (1 << 24)

/* The spherical projection pi_s (grid convention: DESIGN.md reading R1):
 * azimuth phi_i = -pi + (i+1/2) 2pi/W, elevation theta_j = elev_max - (j+1/2)(elev_max-elev_min)/H,
 * beam d = (cos theta cos phi, cos theta sin phi, sin theta); sensor frame x forward, y left, z up. */
typedef struct {
  int32_t H, W;
  float elev_min, elev_max;  /* radians, elev_min < elev_max */
  float r_min, r_max;        /* gates on the surfel-centre range; r_max may be INFINITY */
  float T_ws[12];            /* row-major 3x4 [R|t], p_world = R p_sensor + t */
} lgs_sensor;

/* Tiles of the sorted lists: LGS_TILE_W columns x LGS_TILE_H rows of pixels, tile_id = tile_row *
 * ceil(W / LGS_TILE_W) + tile_col.  8 x 4 = one pixel per lane of a warp: a LiDAR surfel covers ~7 x 3
 * pixels, so 16 x 16 lists (BASELINE.json's wording for configs[0]) make a pixel walk ~25 entries per
 * entry inside its rect (measured); the list rule itself does not depend on the tile
 * shape and the CPU list reference takes it as a parameter. */
#define LGS_TILE_W 8
#define LGS_TILE_H 4

/* Bytes of workspace lgs_render_forward / lgs_render_backward need for a map of N
 * surfels, an H x W image and at most max_keys (tile, surfel) pairs. 0 on bad args. */
size_t lgs_workspace_bytes(int64_t N, int32_t H, int32_t W, int64_t max_keys);

/* Forward: steps S1-S5 of SURVEY.md 8(a) (project/cull with explicit 2*pi seam
 * handling + per-tile key counts -> tile ranges -> tile keys (tile_id, range) bucketed by tile ->
 * hand-written per-tile radix sort -> front-to-back compositing with early stop at T < 1e-4).
 *   out_range  [H,W]   D^ = sum_i w_i tau_i   (un-normalised alpha-composited range)
 *   out_alpha  [H,W]   A^ = sum_i w_i = 1 - T_final
 *   out_normal [3,H,W] N^ = sum_i w_i n_i^f  (sensor frame, facing the sensor); may be NULL
 * `workspace` (device, >= lgs_workspace_bytes, 256-byte aligned) is overwritten and is
 * what lgs_render_backward / lgs_query / lgs_debug_tile_lists read afterwards. */
lgs_status lgs_render_forward(const lgs_gaussians* g, const lgs_sensor* s, void* workspace, size_t workspace_bytes,
                              int64_t max_keys, float* out_range, float* out_alpha, float* out_normal,
                              lgs_stream stream);

/* Backward: steps S7-S8.  Needs the workspace exactly as the matching forward call left
 * it (same g, s, max_keys, same stream or properly ordered).  Upstream gradients
 * dL_drange [H,W], dL_dalpha [H,W] (NULL = 0), dL_dnormal [3,H,W] (NULL = 0).
 * Outputs g_mean [N,3], g_quat [N,4] (through the normalisation of q), g_scale [N,2],
 * g_opacity [N].  accumulate = 0: every one of the N rows is overwritten (culled
 * surfels get zeros); accumulate = 1: gradients are added (mapping batches). */
lgs_status lgs_render_backward(const lgs_gaussians* g, const lgs_sensor* s, void* workspace, size_t workspace_bytes,
                               int64_t max_keys, const float* dL_drange, const float* dL_dalpha,
                               const float* dL_dnormal, float* g_mean, float* g_quat, float* g_scale,
                               float* g_opacity, int accumulate, lgs_stream stream);

/* ---- One-launch batched keyframes (the cost of a mapping iteration grows
 * with the map and the keyframes rendered against it).  F <= LGS_MAX_FRAMES keyframes that share the grid (H, W,
 * elevations, range gates: those of s[0]) and differ in pose are rendered against one map by ONE sequence of
 * kernels: the frame index is folded into the tile id (F * n_tiles lists), one projection over F * N (frame,
 * surfel) pairs, one sort, one compositing grid; the backward adds the F frames' gradients per surfel in frame
 * order (the sum of the per-frame losses, R18), so the result equals F calls of lgs_render_forward /
 * lgs_render_backward with accumulate = 1 -- lists and images bit for bit, gradients up to the order of the
 * float atomics inside a frame.
 *   s          host array of F sensors (pose T_ws per frame; H, W, elev_*, r_* must agree)
 *   out_range, out_alpha [F,H,W]; out_normal [F,3,H,W] (may be NULL)
 *   dL_drange, dL_dalpha [F,H,W]; dL_dnormal [F,3,H,W]   (the last two may be NULL = 0)
 *   workspace  >= lgs_workspace_bytes_batch(N, H, W, max_keys, F); max_keys bounds the keys of ALL frames together
 * lgs_query reports the totals over the frames. */
#define LGS_MAX_FRAMES 16
size_t lgs_workspace_bytes_batch(int64_t N, int32_t H, int32_t W, int64_t max_keys, int32_t F);
lgs_status lgs_render_forward_batch(const lgs_gaussians* g, const lgs_sensor* s, int32_t F, void* workspace,
                                    size_t workspace_bytes, int64_t max_keys, float* out_range, float* out_alpha,
                                    float* out_normal, lgs_stream stream);
lgs_status lgs_render_backward_batch(const lgs_gaussians* g, const lgs_sensor* s, int32_t F, void* workspace,
                                     size_t workspace_bytes, int64_t max_keys, const float* dL_drange,
                                     const float* dL_dalpha, const float* dL_dnormal, float* g_mean, float* g_quat,
                                     float* g_scale, float* g_opacity, int accumulate, lgs_stream stream);

/* Loss stage S6: L = L_depth + lambda_n (lambda_ng L_ng + lambda_ns L_ns) over the valid
 * set Omega_M = {target_range > 0 and keep_mask != 0} (Eq. 10 left, Eq. 11).
 *   target_normal [3,H,W] sensor frame, zero where unknown (M_N); NULL = no L_ng
 *   keep_mask     [H,W] uint8 reliability mask, 0 drops the pixel; NULL = keep all
 *   detach_surf   != 0: N_surf is treated as a constant (no gradient into D^ through it)
 *   loss          device float[4]: L, L_depth, L_ng, L_ns
 *   dL_drange, dL_dalpha [H,W], dL_dnormal [3,H,W]: overwritten (dL_dalpha = 0: the opacity
 *   loss L_alpha of Eq. 10 is outside this call).
 * loss_workspace: device, 8-byte aligned, >= lgs_loss_workspace_bytes(H, W), overwritten (counters and the
 * per-column / per-row beam table).
 * Ordering: plain stream order, as for every call of this library -- including two loss calls in a row on the same
 * loss_workspace and gradient images.  (Inside, the first kernel is launched with programmatic stream serialisation so
 * that its reads of the targets overlap the tail of whatever precedes it; it writes nothing before its
 * griddepcontrol.wait, and like every kernel this library launches that way it executes that wait before it retires, so
 * whatever follows it in the stream is ordered behind everything that precedes it -- DESIGN.md section 1.) */
size_t lgs_loss_workspace_bytes(int32_t H, int32_t W);
lgs_status lgs_loss_range_normal(const lgs_sensor* s, const float* range, const float* alpha, const float* normal,
                                 const float* target_range, const float* target_normal, const uint8_t* keep_mask,
                                 float lambda_n, float lambda_ng, float lambda_ns, int detach_surf,
                                 void* loss_workspace, size_t loss_workspace_bytes, float* loss,
                                 float* dL_drange, float* dL_dalpha, float* dL_dnormal, lgs_stream stream);

/* Loss stage of the full mapping objective, image side of Eq. 13:
 *   L = L_depth + lambda_alpha L_alpha + lambda_n (lambda_ng L_ng + lambda_ns L_ns),
 * L_alpha = -(1/|Omega_M|) sum_{Omega_M} log(A^ + alpha_eps)  (Eq. 10 right: positive-only
 * BCE(A^, 1)); everything else as lgs_loss_range_normal.  Differences: `alpha` [H,W] is read,
 * dL_dalpha = -lambda_alpha / (|Omega_M| (A^ + alpha_eps)) on Omega_M (0 elsewhere), and
 * loss is a device float[5]: L, L_depth, L_ng, L_ns, L_alpha.  The paper's weights are lambda_alpha = 0.1,
 * lambda_n = 1, lambda_ng = 0.05, lambda_ns = 0.01; alpha_eps is not printed (R20). */
lgs_status lgs_loss_mapping(const lgs_sensor* s, const float* range, const float* alpha, const float* normal,
                            const float* target_range, const float* target_normal, const uint8_t* keep_mask,
                            float lambda_alpha, float alpha_eps, float lambda_n, float lambda_ng, float lambda_ns,
                            int detach_surf, void* loss_workspace, size_t loss_workspace_bytes, float* loss,
                            float* dL_drange, float* dL_dalpha, float* dL_dnormal, lgs_stream stream);

/* Optimiser step that closes the mapping iteration: one Adam step on
 * Theta = {mu, q, s~, alpha} with s~ = log s, fused with the scale regulariser
 * L_scale = sum_i max(0, max(s_i0, s_i1) - s_max) (Eq. 12) weighted by lambda_s (Eq. 13).
 * Per surfel: s = exp(s~); g_s += lambda_s dL_scale/ds (even split at s0 == s1); g_s~ = s g_s; then for each
 * of the 10 components  m <- b1 m + (1-b1) g,  v <- b2 v + (1-b2) g^2,
 * theta <- theta - lr (m / (1 - b1^t)) / (sqrt(v / (1 - b2^t)) + eps);  alpha is clipped to
 * [alpha_lo, alpha_hi]; q is not re-normalised (the renderer normalises inside).  The paper names no optimiser:
 * Adam with caller-supplied rates is DESIGN.md reading R21.
 *   mean [N,3], quat [N,4], log_scale [N,2], opacity [N]      parameters, updated in place
 *   scale [N,2]                                               out: exp(new log_scale), what lgs_render_* read
 *   g_mean, g_quat, g_scale, g_opacity                        gradients from lgs_render_backward (activated space)
 *   m, v [N,10]                                               Adam moments (mu 3, q 4, s~ 2, alpha 1), in place
 *   loss_scale                                                device float: L_scale BEFORE the step (overwritten)
 * All device pointers, fp32; `h` is read from host memory at call time; step t >= 1. */
typedef struct {
  float lr_mean, lr_quat, lr_scale, lr_opacity;
  float beta1, beta2, eps;
  int32_t step;
  float lambda_s, s_max;
  float alpha_lo, alpha_hi;
  const int32_t* step_device;  /* optional DEVICE pointer: if not NULL the step count t (>= 1) is read from it when the
                                  kernel runs and `step` is ignored -- a captured CUDA graph that also advances the
                                  counter on the device replays correct bias corrections */
} lgs_adam;
lgs_status lgs_adam_step(int64_t N, float* mean, float* quat, float* log_scale, float* opacity, float* scale,
                         const float* g_mean, const float* g_quat, const float* g_scale, const float* g_opacity,
                         float* m, float* v, const lgs_adam* h, float* loss_scale, lgs_stream stream);

/* Scan -> spherical range image ("we build each scan as a spherical range image
 * ... under the same spherical projection pi_s"): the step that produces the loss stage's targets.
 *   points  [M,3] device fp32, SENSOR frame (a deskewed scan; s->T_ws is not used), metres
 *   normals [M,3] device fp32 or NULL: the tracker's normals N_g-icp
 * Pixel (j, i) owns azimuth [-pi + i dphi, -pi + (i+1) dphi) and elevation (elev_max - (j+1) dth, elev_max - j dth]
 * (the renderer's grid, R1; azimuth +pi wraps to column 0); phi = atan2(y, x), theta = atan2(z, hypot(x, y)),
 * taken in fp64.  Per pixel the nearest return wins (fp32 range; ties: lowest point index); points that are not finite,
 * have range 0 or outside [r_min, r_max], or lie outside the elevation field of view are dropped.
 *   out_range  [H,W]   range of the winner, 0 where no return (M_D = [D > 0])
 *   out_normal [3,H,W] normal of the winner (0 where none or normals == NULL); may be NULL
 *   zbuf       device scratch, 8-byte aligned, >= 8 * H * W bytes, overwritten
 * M <= 2^32 - 1. */
lgs_status lgs_scan_to_range_image(const float* points, const float* normals, int64_t M, const lgs_sensor* s,
                                   void* zbuf, size_t zbuf_bytes, float* out_range, float* out_normal,
                                   lgs_stream stream);

/* The same scan -> range image step for a caller that cannot supply the z-buffer because it cannot allocate device
 * memory where it runs: a per-scan real-time callback that must stay clear of cudaMalloc (a driver lock, possibly a
 * device-wide synchronisation), a process whose device memory was all handed to a pool at start-up, a plugin inside a
 * host program that owns every allocation.  Inputs and outputs are still the caller's; only the scratch is not: the
 * z-buffer is a fixed array of LGS_SCAN_STATIC_MAX_PIXELS 64-bit words (2 MiB) inside the library, which every GPU that
 * loads the library keeps until the process exits.  This call never calls cudaMalloc / cudaFree or anything that does.
 *   - H * W > LGS_SCAN_STATIC_MAX_PIXELS (262,144 = 128 x 2048, the largest image of BASELINE.json's configs) returns
 *     LGS_ERR_STATIC_LIMIT and launches nothing; use lgs_scan_to_range_image with your own buffer for larger grids.
 *   - Every other argument, the result and the error codes are those of lgs_scan_to_range_image (outputs bit for bit).
 *   - The first call on each device looks up where that device holds the array (cudaGetSymbolAddress; this can make the
 *     runtime load the library's GPU code on that device).  Make that first call during start-up, with the device current,
 *     and before any stream capture begins; later calls on that device only launch kernels.
 *   - There is ONE array per GPU and every call on that GPU uses it.  Each call resets the part it uses before writing
 *     it, so calls in sequence (one stream, or streams ordered by events) do not see each other's leftovers; two calls
 *     that may run on the GPU at the same time (different streams, no ordering; different host threads) race on it and
 *     both results are then undefined. */
#define LGS_SCAN_STATIC_MAX_PIXELS (1 << 18)
lgs_status lgs_scan_to_range_image_static(const float* points, const float* normals, int64_t M, const lgs_sensor* s,
                                          float* out_range, float* out_normal, lgs_stream stream);

/* Opacity prune + compaction of the map (first item; "opacity-based pruning",
 * PAPER.md:160, 166 "alpha_min <= alpha_i"): surfel i is kept iff opacity[i] >= alpha_min (NaN: dropped); the
 * survivors keep their relative order; every per-surfel row moves with its surfel.
 *   in : mean [N,3], quat [N,4], log_scale [N,2], opacity [N] (required); scale [N,2], m [N,10], v [N,10] (each may be
 *        NULL together with its output)
 *   out: the same arrays compacted (device, caller-owned, N rows of capacity each, must not overlap the inputs)
 *   n_out: device int64, the number of survivors;  workspace: device, >= lgs_prune_workspace_bytes(N), overwritten.
 * alpha_min is a caller input (the paper prints no value; R28).  All device pointers, fp32. */
size_t lgs_prune_workspace_bytes(int64_t N);
lgs_status lgs_prune_compact(int64_t N, float alpha_min, const float* mean, const float* quat, const float* log_scale,
                             const float* opacity, const float* scale, const float* m, const float* v, float* out_mean,
                             float* out_quat, float* out_log_scale, float* out_opacity, float* out_scale, float* out_m,
                             float* out_v, int64_t* n_out, void* workspace, size_t workspace_bytes, lgs_stream stream);

/* ---- Map management (section 3.3 "Control Score", section 3.5).  Everything the paper
 * leaves open is a caller input; the rules are readings R29-R36 of DESIGN.md section 3.  All data pointers: device, fp32,
 * 16-byte aligned, caller-owned; small parameter arrays / structs are read from HOST memory at call time. ---------------- */

/* Control score, Eq. 9: with lambda_j = sigma_j^2 (sigma [N,3], sorted descending),
 * linear = (l0 - l1) / (l0 + eps), curv = l2 / (l0 + l1 + l2 + eps), x~ = clip((x - lo) / (hi - lo), 0, 1) (R29),
 * c = clip(w_l linear~ + w_c curv~ + w_r res~, 0, 1).  bounds (host) = {lo_l, hi_l, lo_c, hi_c, lo_r, hi_r}, hi > lo;
 * weights (host) = {w_l, w_c, w_r} (the paper's: 0.55, 0.30, 0.15); res [N] G-ICP residuals; c [N] out. */
lgs_status lgs_control_score(int64_t N, const float* sigma, const float* res, const float* bounds, const float* weights,
                             float eps, float* c, lgs_stream stream);

/* Q_q(x) of PAPER.md:160, 166 (R30): the k-th smallest of x [N], k = clip(ceil(q N), 1, N), exact (radix select on the
 * bit patterns: x must be finite and >= 0, as control scores and squared offsets are).  *out (device float) = result
 * (0 if N = 0).  workspace: device, >= lgs_manage_workspace_bytes(N), overwritten. */
size_t lgs_manage_workspace_bytes(int64_t N);
lgs_status lgs_quantile(int64_t N, const float* x, double q, float* out, void* workspace, size_t workspace_bytes,
                        lgs_stream stream);

/* Structure-aware adaptive split (R31, R32).  Candidates: c_i > *thr (device float, e.g. from
 * lgs_quantile with q_split) and opacity_i >= alpha_min; at most max_splits of them split, those of largest c_i (ties:
 * lower index).  A split surfel i becomes two children at mu_i +- shift * s_{i,0} * a_i, a_i = R(q_i) e_0, with both
 * scales divided by `shrink`, q and opacity copied and zero optimiser moments: child "+" overwrites row i, child "-" is
 * appended at row N + (rank of i among the split surfels), so the arrays (updated IN PLACE) must have room for
 * N + max_splits rows.  scale / m / v may be NULL.  flags_out [N] uint8 (may be NULL): 1 = split.
 * *n_new (device int64) = N + number of splits.  workspace >= lgs_manage_workspace_bytes(N). */
lgs_status lgs_split(int64_t N, const float* c, const float* thr, float alpha_min, int64_t max_splits, float shift,
                     float shrink, float* mean, float* quat, float* log_scale, float* opacity, float* scale, float* m,
                     float* v, uint8_t* flags_out, int64_t* n_new, void* workspace, size_t workspace_bytes,
                     lgs_stream stream);

/* One pass of multi-pass planar cover-and-prune (R33-R36).  The means are projected onto world axes
 * (axis_a, axis_b) and grouped in a dense grid of dim_a x dim_b square cells of size `cell` with corner (origin_a,
 * origin_b).  Planar candidates: c_i <= *thr (device float: Q_{q_plane}(c)) and opacity_i >= alpha_min.  Per cell the
 * candidate of largest opacity (ties: lower index) is the representative; with rho^2 the squared offset of another
 * candidate ("member") in the representative's tangent-plane coordinates divided by its scales, the cover radius is
 * R^2 = max(kappa^2, Q_{q_cover}(rho^2 over the cell's members)); the representative's scales (and log_scale, if given)
 * grow by R / kappa, capped at s_max; members with rho^2 <= R^2 are removed -- at most max_removed per pass, lowest
 * indices first.  keep [N] uint8 out: 0 = removed (feed it to lgs_compact); *n_removed: device int64.
 * workspace >= lgs_cover_workspace_bytes(N, dim_a, dim_b).
 * Cost of the grid: the pass keeps per-cell state and visits EVERY cell (one scan over dim_a * dim_b counters by a single
 * CTA, one sort CTA per cell, empty or not), so its time and workspace grow with dim_a * dim_b even when almost all cells are
 * empty.  dim_a * dim_b <= 2^28 is the hard limit (LGS_ERR_INVALID_ARG beyond it); keep the grid within a few times the
 * number of candidates -- crop origin / dims to the candidates' bounding box, or run the pass per map block. */
typedef struct {
  int32_t axis_a, axis_b;
  float origin_a, origin_b, cell;
  int32_t dim_a, dim_b;
  float alpha_min, kappa, q_cover, s_max;
  int64_t max_removed;
} lgs_cover_params;
size_t lgs_cover_workspace_bytes(int64_t N, int32_t dim_a, int32_t dim_b);
lgs_status lgs_cover_prune_pass(int64_t N, const float* mean, const float* quat, float* scale, float* log_scale,
                                const float* opacity, const float* c, const float* thr, const lgs_cover_params* p,
                                uint8_t* keep, int64_t* n_removed, void* workspace, size_t workspace_bytes,
                                lgs_stream stream);

/* Order-preserving compaction by keep flags (what follows a cover-and-prune pass): as lgs_prune_compact, with
 * keep [N] uint8 (0 = drop) instead of the opacity threshold.  workspace >= lgs_prune_workspace_bytes(N). */
lgs_status lgs_compact(int64_t N, const uint8_t* keep, const float* mean, const float* quat, const float* log_scale,
                       const float* opacity, const float* scale, const float* m, const float* v, float* out_mean,
                       float* out_quat, float* out_log_scale, float* out_opacity, float* out_scale, float* out_m,
                       float* out_v, int64_t* n_out, void* workspace, size_t workspace_bytes, lgs_stream stream);

/* Counters of the last forward on this workspace (host outputs; any may be NULL).
 * Synchronises the stream.  Returns LGS_ERR_KEY_OVERFLOW if n_keys > max_keys was hit
 * (n_keys is then the capacity needed). n_contrib = contributing (pixel, surfel) pairs. */
lgs_status lgs_query(const void* workspace, int64_t N, int32_t H, int32_t W, int64_t max_keys, int64_t* n_visible,
                     int64_t* n_keys, int64_t* n_contrib, lgs_stream stream);

/* Test-only: the sorted lists of the last forward on this workspace, unpacked into caller-provided
 * device buffers (any may be NULL): keys_out [n_keys] = tile_id << 32 | float_bits(range key), sorted;
 * vals_out [n_keys] = surfel index; rects_out [N,4] int32 = col_min, ncols (0 = culled), row_min,
 * row_max.  *tile_ranges (host out) = device pointer into the workspace, [n_tiles,2] = [start,end).
 * `s` must be the sensor of that forward.  Synchronises. */
lgs_status lgs_debug_tile_lists(const void* workspace, const lgs_sensor* s, int64_t N, int64_t max_keys,
                                uint64_t* keys_out, uint32_t* vals_out, const uint32_t** tile_ranges,
                                int32_t* rects_out, lgs_stream stream);

/* The same for a batched forward: keys carry the global tile id f * n_tiles + tile, rects_out is [F,N,4],
 * *tile_ranges is [F * n_tiles, 2]. */
lgs_status lgs_debug_tile_lists_batch(const void* workspace, const lgs_sensor* s, int32_t F, int64_t N, int64_t max_keys,
                                      uint64_t* keys_out, uint32_t* vals_out, const uint32_t** tile_ranges,
                                      int32_t* rects_out, lgs_stream stream);

/* Test-only: the hand-written segmented radix sort on its own.  Sorts every segment
 * [seg_ranges[2k], seg_ranges[2k+1]) of (keys, vals) in place by (key, vals) ascending -- the
 * order of a tile list.  tmp_keys / tmp_vals: scratch of the same size as keys / vals. All device. */
lgs_status lgs_debug_segmented_sort(uint32_t* keys, uint32_t* vals, uint32_t* tmp_keys, uint32_t* tmp_vals,
                                    const uint32_t* seg_ranges, int32_t n_segments, lgs_stream stream);

/* Test-only: enabled = 0 launches every kernel in plain stream order (no programmatic dependent launch); 1 (the
 * default) restores the overlapped launches.  Process-wide; results must not depend on it. */
lgs_status lgs_debug_set_pdl(int enabled);

/* Measurement aid: per-kernel device times of the most recent calls, taken with CUDA events
 * recorded on the launching stream around each kernel (or kernel group).  Off by default; when
 * on, calls made while the stream is being captured into a CUDA graph are not instrumented.
 * lgs_profile_read synchronises the stream, writes LGS_PROF_SLOTS durations in milliseconds to the
 * host array `ms` (0 for slots not launched since the last read) and clears them.
 * The events are the only objects the library ever creates (once, on first enable). */
#define LGS_PROF_SLOTS 8
typedef enum {
  LGS_PROF_PROJECT = 0,        /* K1a project / cull / rect / per-tile key counts (+ counter memset) */
  LGS_PROF_EMIT = 1,           /* K1b tile ranges (scan) + K1c key emission bucketed by tile */
  LGS_PROF_SORT = 2,           /* K3 per-tile radix sort */
  LGS_PROF_COMPOSITE_FWD = 3,  /* K5 */
  LGS_PROF_LOSS = 4,           /* K6 (both kernels) */
  LGS_PROF_COMPOSITE_BWD = 5,  /* K7 (+ memset of the partial sums) */
  LGS_PROF_CHAIN = 6,          /* K8 */
  LGS_PROF_ADAM = 7            /* lgs_adam_step */
} lgs_prof_slot;
lgs_status lgs_profile_enable(int on);
lgs_status lgs_profile_read(float* ms, lgs_stream stream);
const char* lgs_profile_slot_name(int slot);

/* Measurement aid: micro-benchmarks behind the roofline denominators (the FP32 and SFU issue peaks
 * are to be confirmed "with an FFMA and a MUFU.EX2 micro-benchmark").  Runs the benchmark
 * `which` on `stream` (best of 5 timed launches after one warm-up, CUDA events), SYNCHRONISES, and writes the rate
 * to *rate_per_s (host): lane-instructions per second for LGS_MB_FFMA / LGS_MB_MUFU_EX2; visits of a 64-byte row per
 * second for the two scatter-add benchmarks (13 scalar red.global.add.f32 per visit against 4 red.global.add.v4.f32;
 * `param` = number of consecutive lanes that share a row, the rows are drawn from scratch_bytes / 64 rows).
 * scratch: device, 16-byte aligned, >= 64 bytes, overwritten.  ms_out (host, may be NULL): duration of the best launch. */
typedef enum { LGS_MB_FFMA = 0, LGS_MB_MUFU_EX2 = 1, LGS_MB_RED_F32 = 2, LGS_MB_RED_F32X4 = 3 } lgs_microbench_kind;
lgs_status lgs_microbench(int which, void* scratch, size_t scratch_bytes, int param, double* rate_per_s,
                          float* ms_out, lgs_stream stream);

/* Library version string (host pointer, static storage). */
const char* lgs_version(void);

#ifdef __cplusplus
}
#endif
#endif /* LGS_H_ */
