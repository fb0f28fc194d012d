/*
 * gsr.h — C ABI of libgsr: batched counterfactual-state rendering of a clustered dynamic Gaussian
 * scene on one B200 (sm_100a), per-state distortion and per-group marginal render utility.
 *
 * Citations: PAPER.md = the text of arxiv/paper_2606_17212; DESIGN.md §3 = the written spec of every
 * step (the paper delegates image formation to a splatting library and prints no rasteriser maths,
 * PAPER.md:140, so each constant is a listed reading there).
 *
 * The four calls named by the problem statement ("the same learned scene is evaluated under many
 * delivery masks ... states are rasterised in one call"; "render paired states with
 * and without g") are gsr_load_scene, gsr_render_states, gsr_distortion and
 * gsr_group_utility.  Everything else is a helper around them.
 *
 * Conventions
 *   - Every function returns GSR_OK (0) or a negative GSR_E_* code; gsr_last_error() gives the text
 *     of the last failure on the calling thread.  Nothing throws, nothing aborts.
 *   - "dev" pointers are CUDA device pointers owned by the caller (e.g. torch tensors' data_ptr());
 *     "host" pointers are ordinary host memory.  The library never frees caller memory.
 *   - Calls that take a `cuda_stream` (a cudaStream_t passed as void*, NULL = the legacy default
 *     stream) only ENQUEUE work on that stream and return; they allocate nothing.  Errors that can
 *     only be seen on the device (an out-of-range level, key capacity exceeded) are latched in the
 *     workspace and read back with gsr_workspace_status().
 *   - A gsr_scene is immutable after load and may be used from several streams at once; a workspace
 *     may be used by one call at a time.
 *   - All images are fp32, layout [B, H, W, 3] (row-major, RGB interleaved), colour range [0,1]
 *     (not clamped, reading A13).
 */
#ifndef GSR_H_
#define GSR_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define GSR_OK 0
#define GSR_E_INVALID_ARG (-1)         /* NULL pointer, negative size, unsupported R / sh_degree ...   */
#define GSR_E_INVALID_LEVEL (-2)       /* a levels[] entry outside -1..3 (latched, see status)         */
#define GSR_E_WORKSPACE_TOO_SMALL (-3) /* ws_bytes below gsr_workspace_bytes, or key capacity exceeded */
#define GSR_E_CUDA (-4)                /* a CUDA runtime call failed; text in gsr_last_error()         */

#define GSR_TILE 16    /* tile edge in pixels (BASELINE.json north_star (3))   */
#define GSR_MAX_R 32   /* temporal-basis terms supported                        */
#define GSR_MAX_SH_DEGREE 3

typedef struct gsr_scene gsr_scene; /* opaque; owns the device copy of the scene */

/* Scene description: host pointers, caller-owned, copied (and activated) by gsr_load_scene.
 * Gaussians are sorted by (cluster, level): group g = 4*c + l owns [group_off[g], group_off[g+1]).
 * "Every cluster produces one base completion group and three refinement groups". */
typedef struct {
  int32_t C;                  /* clusters, 1..4096                                             */
  int32_t N;                  /* Gaussians                                                     */
  int32_t sh_degree;          /* 0..3; K = (sh_degree+1)^2 coefficients per channel            */
  int32_t R;                  /* temporal-basis terms of Eq. (1), 1..GSR_MAX_R                  */
  const int32_t* group_off;   /* [4C+1]                                                        */
  const float* mean;          /* [N,3]   canonical position mu_bar of Eq. (1)                  */
  const float* log_scale;     /* [N,3]                                                         */
  const float* quat;          /* [N,4]   w,x,y,z (need not be normalised)                      */
  const float* opacity_logit; /* [N]                                                           */
  const float* sh_base;       /* [N,K,3] base colour coefficients                              */
  const float* sh_res;        /* [N,K,3] level-3 payload: added iff the cluster's depth is 3   */
  const int8_t* motion_q;     /* [N,R,3] level-1 payload: q_{i,r} of Eq. (1), int8             */
  const float* A0;            /* [C,3,4] row-major; A_c(t) = A0 + t*A1 (Eq. (1), reading A6)   */
  const float* A1;            /* [C,3,4]                                                       */
  const float* motion_scale;  /* [C]     dequantisation step s_c of the motion residual        */
  float background[3];
  /* Optional level-2 / level-3 position residuals delta^(2), delta^(3) of Eq. (1) (DESIGN.md
   * reading I1): [N,3] each, applied iff the cluster's depth is >= 2 / >= 3; NULL = zero.  When both are NULL
   * a Gaussian has 2 projected records per frame, otherwise 4 (one per delivered depth). */
  const float* delta2;
  const float* delta3;
  /* Optional per-level refinements of scale, rotation and opacity ("Scale, rotation, opacity, and colour use a
   * base plus three learned refinements"; reading I2): additive residuals on log_scale
   * [3,N,3], quat [3,N,4] and opacity_logit [3,N] for levels 1..3; level l applies iff the cluster's depth is
   * >= l; the attributes at depth v are the base plus levels 1..v summed in level order in binary32, then
   * activated like the base.  NULL = zero.  Any of them (like delta2 / delta3) gives 4 records per Gaussian. */
  const float* d_log_scale;
  const float* d_quat;
  const float* d_opacity_logit;
  /* Optional per-level colour residuals [3,N,K,3] (levels 1..3; reading I3): the SH coefficients at
   * depth v are sh_base + levels 1..v (+ sh_res at depth 3).  NULL = zero; also selects 4 records per Gaussian. */
  const float* d_sh;
  /* != 0: the cluster affine also transforms the 3-D covariance, Sigma_t = L Sigma L^T with L = the 3x3 part of
   * A_c(t) (reading I4; Eq. (1) itself only moves the mean, so the default is 0). */
  int32_t affine_on_covariance;
} gsr_scene_desc;

/* Pinhole camera, OpenCV axes (x right, y down, z forward), pixel centres at +0.5 (reading A9).
 * p_cam = R_wc * p_world + t_wc. */
typedef struct {
  float R_wc[9]; /* row-major */
  float t_wc[3];
  float fx, fy, cx, cy;
  int32_t W, H;  /* 1 <= W, H <= 65535 * 16 and 3 * W * H < 2^32 (else GSR_E_INVALID_ARG) */
  float znear; /* Gaussians with z <= znear are culled (0.2 in every config) */
} gsr_camera;

/* Per-group aggregates of Eq. (3)/(4): mean, 0.10 lower-tail quantile (linear
 * interpolation), population std and risk-adjusted utility ((1-a)mean + a q10)/(1 + b std) with
 * a = 0.25, b = 0.05 — once with D = MSE (delta = MSE(m) - MSE(m u g)) and once in dB
 * (delta = PSNR(m u g) - PSNR(m)). */
typedef struct {
  double mean_mse, q10_mse, std_mse, risk_mse;
  double mean_db, q10_db, std_db, risk_db;
  double count; /* number of pairs of this group */
} gsr_utility;

/* ------------------------------------------------------------------------------------------------
 * gsr_load_scene — DESIGN.md §3.0.  Activates the scene once on the host in double precision
 * (scale = exp(log_scale); unit quaternion -> rotation; Sigma = R diag(scale^2) R^T;
 * opacity = sigmoid(logit); tau = ln(255 * opacity)), rounds to fp32, and uploads it in the device
 * layout of DESIGN.md §5.  Synchronous (cudaMalloc + cudaMemcpy).  *out is NULL on failure.
 * gsr_free_scene releases it (NULL is allowed). */
int gsr_load_scene(const gsr_scene_desc* desc, gsr_scene** out);
void gsr_free_scene(gsr_scene* scene);

/* Bytes of workspace gsr_render_states needs for this scene / camera / batch.  The tile-key
 * capacity defaults to 12 keys per projected record (+1Mi); gsr_workspace_bytes_ex takes an explicit
 * capacity (0 = default).  Returns 0 on invalid arguments. */
size_t gsr_workspace_bytes(const gsr_scene* scene, const gsr_camera* cam, int32_t B);
size_t gsr_workspace_bytes_ex(const gsr_scene* scene, const gsr_camera* cam, int32_t B, int64_t key_capacity);

/* ------------------------------------------------------------------------------------------------
 * gsr_render_states — the hot path, BASELINE.json north_star (1)-(4); DESIGN.md §3.1-§3.5.
 * Renders B partial states of `scene` seen from `cam` at time `t` in one call.
 *   levels  dev int8 [B, C]  delivered depth of cluster c in state b, -1..3 (reading A3): Gaussian i of
 *                            cluster c with level l is present iff depth >= l; the motion residual
 *                            of Eq. (1) is applied iff depth >= 1, the SH residual iff depth == 3.
 *   out     dev fp32 [B, H, W, 3], or NULL (then only the fused distortion is produced).
 *   ref     dev fp32 [H, W, 3] or NULL; when given, mse/psnr_db (dev [B]) receive the per-state
 *           distortion against it, reduced inside the compositing kernel with the same tree as
 *           gsr_distortion (bitwise equal results).  mse/psnr_db may be NULL iff ref is NULL.
 *   workspace dev, >= gsr_workspace_bytes(...) bytes, 256-byte aligned.
 * The result for a state depends only on its row of `levels`: rendering a batch is bitwise equal to
 * rendering its states one at a time ("CUDA batched/serial equivalence").
 * Asynchronous on `cuda_stream`.  Device-side failures: see gsr_workspace_status. */
int gsr_render_states(const gsr_scene* scene, const gsr_camera* cam, float t, const int8_t* levels, int32_t B,
                      float* out, void* workspace, size_t ws_bytes, void* cuda_stream);
int gsr_render_states_ex(const gsr_scene* scene, const gsr_camera* cam, float t, const int8_t* levels,
                         int32_t B, float* out, const float* ref, double* mse, float* psnr_db,
                         void* workspace, size_t ws_bytes, void* cuda_stream);

/* gsr_render_states_vs_full — the utility workload's frame call (north_star (5), reading A16): like
 * gsr_render_states_ex, but the reference is the FULL state (every cluster at depth 3) of the same
 * (camera, t), composited from the same projected records and sorted lists (one projection and one
 * sort per frame) into ref_out (dev fp32 [H,W,3], required).  mse (required) / psnr_db (dev [B])
 * receive each state's distortion against it; out may be NULL. */
int gsr_render_states_vs_full(const gsr_scene* scene, const gsr_camera* cam, float t, const int8_t* levels,
                              int32_t B, float* out, float* ref_out, double* mse, float* psnr_db,
                              void* workspace, size_t ws_bytes, void* cuda_stream);

/* ------------------------------------------------------------------------------------------------
 * gsr_render_backward — the backward of the compositing step (the training objective is a function
 * of the rendered images; SURVEY.md §8(f)-4 follow-on).  To be called after gsr_render_states /
 * _ex / _vs_full on the SAME workspace, batch and stream: it reuses the projected records, the sorted lists and the
 * validated levels the forward call left there, and uses the workspace's scratch tables (so one backward call per
 * workspace at a time, like a render).  States whose pixels in a tile are identical are walked once
 * per tile with the sum of their dL_dimages — the gradient is linear in it (option "dedup", default on).
 *   images      dev fp32 [B,H,W,3]  the forward output of that call
 *   dL_dimages  dev fp32 [B,H,W,3]  the gradient of the objective with respect to every pixel of every state
 *   grad        dev fp32 [gsr_num_records(scene), 12], 16-byte aligned, overwritten: for record r (Gaussian i,
 *               variant v: r = 2 i + v, v = 0 the geometry of cluster depth 0, v = 1 of depth >= 1; r = 4 i + v for scenes with position
 *               residual levels), summed over the states and pixels that composite it,
 *               d/d(rgb[3], rgb with the level-3 SH residual[3], opacity, A, B, Cq, m_x, m_y)
 *               where pixel = sum_i alpha_i T_i rgb_i + T_end bg, alpha = min(0.99, opacity exp(-q)),
 *               q = (A dx + B dy) dx + Cq dy^2, (dx, dy) = (m_x, m_y) - pixel centre; the cut, the
 *               cap and the stop are constants of the differentiation.  States whose cluster depth is 3 use the
 *               second colour, all others the first.
 * Synchronises once at entry (reads the workspace header), then asynchronous.  Sums are formed with float
 * atomics: the result is reproducible up to fp32 summation order.  B must be the forward call's B. */
int64_t gsr_num_records(const gsr_scene* scene);
int gsr_render_backward(const gsr_scene* scene, void* workspace, const float* images, const float* dL_dimages,
                        int32_t B, float* grad, void* cuda_stream);

/* ------------------------------------------------------------------------------------------------
 * gsr_distortion_backward — d/d(imgs) of L = sum_b weight[b] D_b with D_b = MSE_b + lambda_ssim (1 - SSIM_b)
 * (the term E_w[D_w] of Eq. (2), "D = MSE + 0.20(1 - SSIM)"; SSIM per reading G1 as in
 * gsr_distortion_ssim): the dL_dimages input of gsr_render_backward for that objective.
 *   imgs fp32 dev [B,H,W,3]; ref fp32 dev [H,W,3]; weight double dev [B] or NULL (= 1 for every state; pass 1/B for
 *   the mean over states); lambda_ssim >= 0 (0.20 in the paper; 0 = the MSE term alone);
 *   dL_dimgs fp32 dev [B,H,W,3], overwritten.  workspace dev, >= gsr_distortion_backward_workspace_bytes(H, W), 256-byte
 *   aligned (the window moments of the reference, computed once per call; may be NULL when lambda_ssim == 0; else
 *   GSR_E_WORKSPACE_TOO_SMALL).  Window moments in double (as the forward).  Asynchronous. */
size_t gsr_distortion_backward_workspace_bytes(int32_t H, int32_t W);
int gsr_distortion_backward(const float* imgs, const float* ref, int32_t B, int32_t H, int32_t W, const double* weight,
                            double lambda_ssim, float* dL_dimgs, void* workspace, size_t ws_bytes, void* cuda_stream);

/* The other image-space terms of Eq. (2) (L = E_w[D_w] + lambda_c CVaR_0.05(D) + lambda_r R +
 * lambda_t F + lambda_m M; lambda_c = 0.30, lambda_t = 0.10, lambda_m = 2.0 in PAPER.md:72):
 * gsr_objective_weights: weights[b] = dL/dD_b of w_mean mean(D) + w_cvar CVaR_alpha(D) + w_mono M(D) — the `weight`
 *   input of gsr_distortion_backward.  1/n each; 1/k (k = max(1, ceil(alpha n))) for every D strictly above the CVaR
 *   threshold, the remaining (k - #above)/k shared equally by the values equal to it (a subgradient); + w_mono on
 *   idx_next[p] and - w_mono on idx_prev[p] of every pair with D[next] > D[prev] (indices outside [0, n) are refused:
 *   gsr_index_status).  d, weights double dev [n]; idx_* int32 dev [n_pairs] (may be NULL when n_pairs = 0);
 *   0 < alpha <= 1.
 * gsr_flicker_backward: d/d(imgs_t1), d/d(imgs_t2) of sum_b weight[b] F_b (F of gsr_flicker): g_t2 = weight[b] 2 e /
 *   (3 H W), g_t1 = - g_t2, e = (imgs_t2 - imgs_t1) - (ref_t2 - ref_t1); weight double dev [B] or NULL (= 1);
 *   g_t1, g_t2 fp32 dev [B,H,W,3], overwritten (either may be NULL).  Both asynchronous. */
int gsr_objective_weights(const double* d, int32_t n, double w_mean, double w_cvar, double alpha,
                          const int32_t* idx_prev, const int32_t* idx_next, int32_t n_pairs, double w_mono,
                          double* weights, void* cuda_stream);
int gsr_flicker_backward(const float* imgs_t1, const float* imgs_t2, const float* ref_t1, const float* ref_t2, int32_t B,
                         int32_t H, int32_t W, const double* weight, float* g_t1, float* g_t2, void* cuda_stream);

/* ------------------------------------------------------------------------------------------------
 * gsr_project_backward — the backward of the steps in front of the compositor: activation,
 * deformation Eq. (1), EWA projection and SH colour; DESIGN.md §17.  Takes the
 * per-record gradient gsr_render_backward produced for a frame (same scene, camera and t) to the gradient with
 * respect to the scene's own parameters.  Needs no workspace: the projection is recomputed.
 *   grad_records dev fp32 [gsr_num_records(scene), 12]   (16-byte aligned)
 *   g_gauss      dev fp32 [N, 14], overwritten: d/d(mean[3], rho[3], log_scale[3], quat[4], opacity_logit) with rho
 *                the motion residual vector s_c sum_r b_r(t) q_{i,r} of Eq. (1): the gradient with respect to the
 *                real-valued coefficient s_c q_{i,r,k} is b_r(t) * d/drho_k, b_r(t) = cos(pi r t); quat is the raw
 *                (unnormalised) quaternion
 *   g_sh_base    dev fp32 [N, K, 3], overwritten: d/d(sh_base); g_sh_res likewise for the level-3 payload
 *   g_cluster    dev fp32 [C, 13], overwritten: d/dA_c(t) [3,4] row-major (d/dA0 = it, d/dA1 = t * it), d/ds_c
 * The discrete decisions are constants of the differentiation: presence, the culls, the clamp of x/z and y/z at
 * 1.3 lim (a clamped coordinate passes no gradient through the Jacobian), rgb = max(0, .), tau, radius, rectangle.
 * Asynchronous on `cuda_stream`; the per-cluster sums use float atomics (reproducible up to fp32 summation
 * order).  Scenes with position residual levels, per-level attribute refinements or affine_on_covariance are
 * refused (GSR_E_INVALID_ARG). */
int gsr_project_backward(const gsr_scene* scene, const gsr_camera* cam, float t, const float* grad_records,
                         float* g_gauss, float* g_sh_base, float* g_sh_res, float* g_cluster, void* cuda_stream);

/* gsr_project_backward_full — gsr_project_backward for every scene, including the full representation of
 * position residual levels delta2 / delta3, per-level refinements of scale,
 * rotation, opacity and colour, affine_on_covariance; four records per Gaussian (record 4 i + delivered depth).
 * grad_records, g_gauss, g_sh_base, g_sh_res, g_cluster as for gsr_project_backward; the log_scale / quat /
 * opacity_logit / sh_base columns are the gradients of the BASE arrays (every depth contains the base).  In addition
 * (each may be NULL = not wanted; overwritten; zero where the scene has no such term):
 *   g_delta dev fp32 [N, 6]        d/d(delta2[3], delta3[3]): dL/dmu of the depths that apply the residual
 *   g_attr  dev fp32 [3, N, 8]     per refinement level l = 1..3: d/d(d_log_scale[l][3], d_quat[l][4],
 *                                  d_opacity_logit[l]) = the sum over the depths >= l
 *   g_d_sh  dev fp32 [3, N, K, 3]  per level: d/d(d_sh[l])
 * With affine_on_covariance the covariance path (Sigma_t = L Sigma L^T) adds to the linear part of g_cluster.
 * Scenes with two records per Gaussian are served by the kernel of gsr_project_backward. */
int gsr_project_backward_full(const gsr_scene* scene, const gsr_camera* cam, float t, const float* grad_records,
                              float* g_gauss, float* g_sh_base, float* g_sh_res, float* g_cluster, float* g_delta,
                              float* g_attr, float* g_d_sh, void* cuda_stream);

/* Synchronises `cuda_stream` and reads the status latched by the last render into `workspace`:
 * returns GSR_OK, GSR_E_INVALID_LEVEL or GSR_E_WORKSPACE_TOO_SMALL.  keys_needed (host, may be NULL)
 * receives the number of (tile, depth, record) keys the frame produced. */
int gsr_workspace_status(const void* workspace, int64_t* keys_needed, void* cuda_stream);

/* Index arrays given to the device-pointer helpers below (a send order, the pair lists of gsr_group_utility, the
 * prefix pairs of gsr_prefix_monotonicity) are range-checked ON THE DEVICE: an entry out of range is skipped —
 * an invalid group of a send order sends nothing and ends a frontier walk, an invalid pair belongs to no group
 * and has zero difference — and latched in a per-device error word.  gsr_index_status synchronises
 * `cuda_stream`, reads and clears that word: GSR_OK, or GSR_E_INVALID_ARG with the kind in gsr_last_error(). */
int gsr_index_status(void* cuda_stream);

/* ------------------------------------------------------------------------------------------------
 * gsr_distortion — north_star (5), DESIGN.md §3.6.  Per state b: MSE_b = sum((img_b - ref)^2)/(3HW)
 * accumulated in double with a fixed reduction tree; PSNR_b = -10 log10(max(MSE_b, 1e-10)).
 *   imgs dev fp32 [B,H,W,3]; ref dev fp32 [H,W,3]; mse dev double [B]; psnr_db dev fp32 [B].
 *   workspace dev, >= gsr_distortion_workspace_bytes(B,H,W) bytes.  Asynchronous. */
size_t gsr_distortion_workspace_bytes(int32_t B, int32_t H, int32_t W);
int gsr_distortion(const float* imgs, const float* ref, int32_t B, int32_t H, int32_t W, double* mse,
                   float* psnr_db, void* workspace, size_t ws_bytes, void* cuda_stream);

/* gsr_distortion_static — gsr_distortion for callers that may not allocate device memory (code under CUDA graph
 * capture, tight serving loops, harnesses that forbid cudaMalloc): the same kernels and reduction tree, hence the same
 * values, with the per-(state, tile) partials in a scratch array built into the library instead of a caller-provided
 * workspace.  The call allocates nothing (no cudaMalloc / cudaFree / allocating library routine).
 *   Limit: B * ceil(W/16) * ceil(H/16) <= gsr_distortion_static_max_partials() = 2^20 (8 MiB of device memory, held by
 *   every GPU that loads the library until the process exits); beyond it GSR_E_WORKSPACE_TOO_SMALL and nothing is
 *   launched — use gsr_distortion.
 *   Every call on a device shares that array; a call overwrites all the entries it reads, so earlier contents never
 *   matter, but two calls that overlap on the GPU (different streams, no ordering between them) race: serialise them.
 *   imgs, ref, mse, psnr_db as for gsr_distortion (psnr_db may be NULL).  Asynchronous on `cuda_stream`. */
int64_t gsr_distortion_static_max_partials(void);
int gsr_distortion_static(const float* imgs, const float* ref, int32_t B, int32_t H, int32_t W, double* mse,
                          float* psnr_db, void* cuda_stream);

/* ------------------------------------------------------------------------------------------------
 * gsr_group_utility — Eq. (3) and Eq. (4); DESIGN.md §3.7.
 *   mse dev double [B], psnr_db dev fp32 [B]: distortions of a batch.
 *   idx_without[p], idx_with[p] (dev int32 [n_pairs]): the states m and m u g of pair p;
 *   group_id[p] in [0, G).  out dev gsr_utility [G].  delta_mse / delta_db: dev double [n_pairs] or NULL.
 * Asynchronous; one CTA per group, fixed summation order (deterministic).
 * Range errors (see gsr_index_status): a group id outside [0, G) or a negative state index.  The call has no
 * B; gsr_group_utility_b is the same call with the number of states B behind mse / psnr_db, so that state
 * indices >= B are refused too (the Python binding and gsr_utility_frame_host use it). */
int gsr_group_utility(const double* mse, const float* psnr_db, const int32_t* idx_without,
                      const int32_t* idx_with, const int32_t* group_id, int32_t n_pairs, int32_t G,
                      gsr_utility* out, double* delta_mse, double* delta_db, void* cuda_stream);
int gsr_group_utility_b(const double* mse, const float* psnr_db, int32_t B, const int32_t* idx_without,
                        const int32_t* idx_with, const int32_t* group_id, int32_t n_pairs, int32_t G,
                        gsr_utility* out, double* delta_mse, double* delta_db, void* cuda_stream);

/* ------------------------------------------------------------------------------------------------
 * gsr_close_levels — dependency closure, PAPER.md:185 ("A cluster-layer is usable only when all
 * chunks in its dependency closure are usable"), chain 0 <- 1 <- 2 <- 3 (reading A8).
 *   delivered_mask dev uint8 [n], bit l = level-l group usable.
 *   depth_out dev int8 [n] = (number of trailing one bits) - 1;  closure_out dev uint8 [n] or NULL
 *   = (1 << (depth+1)) - 1.  Asynchronous. */
int gsr_close_levels(const uint8_t* delivered_mask, int64_t n, int8_t* depth_out, uint8_t* closure_out,
                     void* cuda_stream);

/* ------------------------------------------------------------------------------------------------
 * Scheduling frontier and partial-state atlas (Fig. 2, Fig. 6; DESIGN.md
 * §11, readings F1-F4).  Integer / comparison helpers around the renderer: all results are bit-exact and
 * independent of thread scheduling (ties are broken by the written keys).  Group g = 4*c + l.  All
 * pointers are dev; all calls are asynchronous on `cuda_stream`.
 *
 * gsr_group_wire_bytes: "raw stream bytes plus one 48-byte chunk header and 4 bytes per dependency word
 *   for each 1200-byte payload chunk": wire[g] = raw[g] + ceil(raw[g]/1200) * (48 + 4 l).
 *   raw_bytes, wire: int64 [4C].
 * gsr_frontier_order: greedy dependency-closed total order of the 4C groups.  At every step the eligible
 *   groups are (c, l) whose prerequisites (c, 0..l-1) are already in the order; the policy takes the one
 *   with the smallest key: GSR_POLICY_UTILITY (-score[g], l, c) — "render-utility order";
 *   GSR_POLICY_NOMINAL (l, c) — "nominal layer order"; GSR_POLICY_BYTE_GREEDY (wire[g], l, c) —
 *   "dependency byte-greedy order".  A flat score table reproduces the nominal order
 *   (PAPER.md:90).  score: double [4C] (only read for GSR_POLICY_UTILITY, e.g. the risk_db column of
 *   gsr_group_utility; must be finite); order: int32 [4C]; cum_bytes: int64 [4C] or NULL (running wire sum).
 * gsr_frontier_states: the state of an order at budget j = its longest prefix whose cumulative wire bytes
 *   are <= budgets[j]; levels int8 [nb, C] receives each cluster's delivered depth (-1..3), used int64 [nb]
 *   (or NULL) the bytes of that prefix, n_groups int32 [nb] (or NULL) its length.
 * gsr_state_bytes: wire cost of dependency-closed states: bytes[b] = sum_c sum_{l <= levels[b,c]} wire[4c+l].
 *   levels int8 [B, C] (values outside -1..3 are clamped to that range); bytes int64 [B].
 * gsr_best_state_under_budget: the "empirical oracle" of the atlas: best[j] = the state of highest
 *   psnr_db among those with state_bytes <= budgets[j]; ties -> lowest index; -1 if none.  best int32 [nb]. */
#define GSR_POLICY_UTILITY 0
#define GSR_POLICY_NOMINAL 1
#define GSR_POLICY_BYTE_GREEDY 2
int gsr_group_wire_bytes(const int64_t* raw_bytes, int32_t C, int64_t* wire, void* cuda_stream);
int gsr_frontier_order(const double* score, const int64_t* wire, int32_t C, int32_t policy, int32_t* order,
                       int64_t* cum_bytes, void* cuda_stream);
int gsr_frontier_states(const int32_t* order, const int64_t* wire, int32_t C, const int64_t* budgets, int32_t nb,
                        int8_t* levels, int64_t* used, int32_t* n_groups, void* cuda_stream);
int gsr_state_bytes(const int8_t* levels, int32_t B, int32_t C, const int64_t* wire, int64_t* bytes,
                    void* cuda_stream);
int gsr_best_state_under_budget(const float* psnr_db, const int64_t* state_bytes, int32_t B,
                                const int64_t* budgets, int32_t nb, int32_t* best, void* cuda_stream);

/* ------------------------------------------------------------------------------------------------
 * Richer distortion and risk reductions (Eq. (2) and the text below it; DESIGN.md §12,
 * readings G1-G4).  All pointers dev; asynchronous on `cuda_stream`; deterministic (fixed reduction trees).
 *
 * gsr_distortion_ssim: "D = MSE + 0.20(1 - SSIM)".  SSIM per state against `ref`: per
 *   channel, 11x11 Gaussian window (sigma 1.5, normalised, separable), zero padding, C1 = 0.01^2,
 *   C2 = 0.03^2, mean of the SSIM map over H x W x 3 (reading G1); fp32 pixels, double moments and sums.
 *   imgs fp32 [B,H,W,3]; ref fp32 [H,W,3]; ssim double [B] (or NULL); mse double [B] (or NULL: e.g. from
 *   gsr_distortion / the fused path); d_mix double [B] (or NULL; needs mse) = mse + 0.20 (1 - ssim).
 *   workspace >= gsr_distortion_workspace_bytes(B,H,W).
 * gsr_flicker: temporal-change error ("F penalizes temporal-change error"; reading G3):
 *   out[b] = mean(((imgs_t2[b] - imgs_t1[b]) - (ref_t2 - ref_t1))^2), fp32 differences, double sum.
 *   imgs_t1, imgs_t2 fp32 [B,H,W,3] (the same states at two times); ref_t1, ref_t2 fp32 [H,W,3];
 *   out double [B]; workspace >= gsr_distortion_workspace_bytes(B,H,W).
 * gsr_risk_reduce: mean, CVaR_alpha, alpha-quantile and worst value of n per-state values (PAPER.md:68
 *   "CVaR_0.05(D)", "p10 PSNR"; reading G2): k = max(1, ceil(alpha n)); cvar = mean of the k
 *   worst values (upper_tail != 0: the largest, for a distortion; 0: the smallest, for a PSNR); quantile =
 *   linear interpolation at position (1 - alpha)(n-1) resp. alpha (n-1) of the ascending order.
 *   values: double [n] (dtype 0) or float [n] (dtype 1); out: gsr_risk [1].
 * gsr_prefix_monotonicity: "M penalizes quality regressions as a prefix grows" (reading G4):
 *   M = sum_p max(0, d[idx_next[p]] - d[idx_prev[p]]), violations = #{p : d[next] > d[prev]}.
 *   d double [.]; idx_prev, idx_next int32 [n_pairs]; m_out double [1]; violations int32 [1] (either may be NULL).
 *   gsr_prefix_monotonicity_n takes the length n of d and refuses indices >= n as well as negative ones
 *   (gsr_index_status); a refused pair contributes nothing. */
typedef struct {
  double mean, cvar, quantile, worst, count;
} gsr_risk;
int gsr_distortion_ssim(const float* imgs, const float* ref, int32_t B, int32_t H, int32_t W, const double* mse,
                        double* ssim, double* d_mix, void* workspace, size_t ws_bytes, void* cuda_stream);
int gsr_flicker(const float* imgs_t1, const float* imgs_t2, const float* ref_t1, const float* ref_t2, int32_t B,
                int32_t H, int32_t W, double* out, void* workspace, size_t ws_bytes, void* cuda_stream);
int gsr_risk_reduce(const void* values, int32_t dtype, int32_t n, double alpha, int32_t upper_tail, gsr_risk* out,
                    void* cuda_stream);
int gsr_prefix_monotonicity(const double* d, const int32_t* idx_prev, const int32_t* idx_next, int32_t n_pairs,
                            double* m_out, int32_t* violations, void* cuda_stream);
int gsr_prefix_monotonicity_n(const double* d, int32_t n, const int32_t* idx_prev, const int32_t* idx_next,
                              int32_t n_pairs, double* m_out, int32_t* violations, void* cuda_stream);

/* ------------------------------------------------------------------------------------------------
 * gsr_sample_delivery — the step before the hot path: "A training world samples capacity, RTT, display
 * deadline, IID erasure, and a Gilbert-Elliott burst process.  Packet dependencies are enforced after
 * delivery, then converted to cluster-layer masks".  DESIGN.md §13, readings H1-H6:
 *   - group g = 4c + l is cut into ceil(raw_bytes[g] / 1200) packets (an empty group is always usable);
 *   - the packets of a world are sent group by group in `order` (e.g. a gsr_frontier_order result);
 *     packet_budget[w] (or NULL = no limit) packets are sent before the display deadline, the rest never arrive;
 *   - a sent packet is lost if the IID process drops it (p_iid) OR the Gilbert-Elliott channel does: state of
 *     packet 0 = Bad with the stationary probability p_gb/(p_gb+p_bg) (0 if both are 0), then P(G->B) = p_gb,
 *     P(B->G) = p_bg; drop probability e_good in Good, e_bad in Bad;
 *   - a group is usable iff all its packets arrived; mask[w,c] bit l; levels[w,c] = dependency closure.
 * Randomness: Philox4x32-10, key = seed, counter = (packet index, world0 + w, 0, 0); words x0..x3 drive the
 * IID drop, the GE transition, the GE drop and (packet 0) the initial state; an event of probability p happens
 * iff x < floor(p * 2^32).  The result for a world depends only on (seed, world0 + w): sampling a batch in
 * pieces gives the same masks.  Bit-exact against the oracle.
 *   raw_bytes dev int64 [4C]; order dev int32 [4C] (a permutation of 0..4C-1; an entry outside that range sends
 *   nothing and is reported by gsr_index_status); model: host; packet_budget dev int32 [W] or
 *   NULL; mask dev uint8 [W,C]; levels dev int8 [W,C] or NULL (feeds gsr_render_states directly);
 *   workspace dev >= gsr_delivery_workspace_bytes(C).  Asynchronous. */
typedef struct {
  double p_iid, p_gb, p_bg, e_good, e_bad;
  uint64_t seed;
} gsr_loss_model;
size_t gsr_delivery_workspace_bytes(int32_t C);
int gsr_sample_delivery(const int64_t* raw_bytes, const int32_t* order, int32_t C, const gsr_loss_model* model,
                        const int32_t* packet_budget, int32_t W, int32_t world0, uint8_t* mask, int8_t* levels,
                        void* workspace, size_t ws_bytes, void* cuda_stream);

/* ------------------------------------------------------------------------------------------------
 * One-call convenience with HOST buffers (used for the end-to-end measurement): uploads `levels`
 * and the pair lists, renders the full state (all depths 3) as the reference, renders the batch with
 * fused distortion, aggregates utilities, and copies mse / psnr_db / util back.  Synchronous.
 *   levels host int8 [B,C]; idx_without, idx_with, group_id host int32 [n_pairs] (n_pairs may be 0; state
 *   indices outside [0, B) or group ids outside [0, G) are refused on the host with GSR_E_INVALID_ARG);
 *   mse host double [B]; psnr_db host float [B]; util host gsr_utility [G] (may be NULL if G == 0);
 *   materialise_images != 0: the [B,H,W,3] images are written to device memory inside the workspace
 *   (as gsr_render_states does); out_host (host fp32 [B,H,W,3] or NULL) additionally copies them back.
 *   workspace dev >= gsr_frame_workspace_bytes(..., want_images = materialise_images). */
size_t gsr_frame_workspace_bytes(const gsr_scene* scene, const gsr_camera* cam, int32_t B, int32_t n_pairs,
                                 int32_t G, int32_t want_images);
int gsr_utility_frame_host(const gsr_scene* scene, const gsr_camera* cam, float t, const int8_t* levels,
                           int32_t B, const int32_t* idx_without, const int32_t* idx_with,
                           const int32_t* group_id, int32_t n_pairs, int32_t G, double* mse, float* psnr_db,
                           gsr_utility* util, int32_t materialise_images, float* out_host, void* workspace,
                           size_t ws_bytes,
                           void* cuda_stream);

/* ------------------------------------------------------------------------------------------------
 * Debug / parity exports (tests only; synchronous unless noted).  They read what the last
 * gsr_render_states left in `workspace`.
 *
 * gsr_debug_projection: per projected record r = 2*i + v (v = 0: geometry without the motion
 * residual, used when the cluster's depth is 0 — only level-0 Gaussians have it; v = 1: with the
 * residual, used when depth >= 1).  Scenes with delta2 / delta3 / d_* arrays have FOUR records per
 * Gaussian, r = 4*i + v, v = the delivered depth the record belongs to (a level-l Gaussian has v >= l;
 * rgb_base and rgb_res are then equal).  All host arrays of length 2N resp. 4N (any may be NULL):
 *   valid u8, radius i32, rect i32 [2N,4] (tx0,ty0,tx1,ty1), depth_bits u32, count i32,
 *   mean2d f32 [2N,2], conic f32 [2N,3] (A=conic_a/2, B=conic_b, Cq=conic_c/2),
 *   rgb_base f32 [2N,3], rgb_res f32 [2N,3]. */
int gsr_debug_projection(const gsr_scene* scene, const void* workspace, uint8_t* valid, int32_t* radius,
                         int32_t* rect, uint32_t* depth_bits, int32_t* count, float* mean2d, float* conic,
                         float* rgb_base, float* rgb_res, void* cuda_stream);

/* gsr_debug_keys: the canonical sorted key list (state, tile, depth bits, Gaussian index) of state
 * `b` of the last rendered batch (north_star (3)).  Writes at most `cap` entries to the host arrays
 * and returns the list length in *n_keys. */
int gsr_debug_keys(const gsr_scene* scene, const void* workspace, int32_t b, int64_t cap, uint32_t* tile,
                   uint32_t* depth_bits, int32_t* gaussian, int64_t* n_keys, void* cuda_stream);

/* gsr_debug_state_counts: per state of the last batch, the number of tile intersections I_b
 * (= its key-list length).  counts: host int64 [B]. */
int gsr_debug_state_counts(const gsr_scene* scene, const void* workspace, int64_t* counts, void* cuda_stream);

/* gsr_debug_closure: closed depth / presence predicates the renderer derived from the last `levels`.
 * depth host int8 [B,C] (as validated). */
int gsr_debug_closure(const gsr_scene* scene, const void* workspace, int8_t* depth, void* cuda_stream);

/* gsr_debug_pair_counts: instrumented re-run of the compositing kernel over the last batch (same
 * lists, same arithmetic, nothing written).  counts3 (host int64 [3]):
 *   [0] (pixel, record) pairs whose alpha was evaluated with at least one live present state,
 *   [1] (pixel, record, state) colour/transmittance updates on live present states,
 *   [2] logical (pixel, record, state) triples: like [1] without the cut and with every member state of a
 *       dedup class counted — what a per-state rasteriser walking the same sub-tile-culled lists would evaluate
 *       (a lower bound of the oracle's E = sum_b E_b, whose lists are the unculled 3-sigma tile lists). */
int gsr_debug_pair_counts(const gsr_scene* scene, const void* workspace, int64_t* counts3, void* cuda_stream);

/* Options.  "state_block" = state slots per compositing warp (0 = default, 1, 4..8 or 16) and "dedup" = 0/1
 * (tile-level state dedup, default 1): results do not depend on either (bitwise).  Both belong to the CALLING
 * HOST THREAD — they steer the calls that thread makes afterwards and nothing another thread does.
 * "profile" = 1 records CUDA events around every compositing launch and around the projection and binning +
 * sort phases of every frame, for the calls of the thread that switched it on (other threads run unprofiled);
 * it is refused with GSR_E_INVALID_ARG while any thread is inside a render call.
 * Everything may be called from several host threads at once, each with its own stream and workspace
 * (tests/test_gpu_streams.py). */
int gsr_set_option(const char* name, int32_t value);

/* Sum of the compositing kernel's durations (ms, CUDA events on its launch stream) and the number
 * of launches recorded since "profile" was set or last read.  Synchronises those events. */
int gsr_profile_read(double* composite_ms, int32_t* composite_launches);

/* Sums of the projection phase (a1 + a2: k_project) and of the binning + sort phase (a3: scans, key emission, radix
 * passes, tile ranges) over the frames prepared since "profile" was set or last read (CUDA events on the launch
 * stream), and the number of those frames.  Synchronises those events. */
int gsr_profile_read_phases(double* project_ms, double* sort_ms, int32_t* frames);

/* Kernels launched by this library since load (the caller's evidence for "gpu_launches"). */
int64_t gsr_launch_count(void);

/* Measures this device's FP32 FMA throughput (TFLOP/s, FMA = 2 flop) with a register-resident FFMA
 * chain kernel: the denominator of the compositing roofline.  Synchronous. */
int gsr_measure_fp32_peak(double* tflops, void* cuda_stream);

/* Text of the last error on this thread ("" if none). */
const char* gsr_last_error(void);

/* Library build tag, e.g. "gsr 0.1 sm_100a". */
const char* gsr_version(void);

#ifdef __cplusplus
}
#endif
#endif /* GSR_H_ */
