// gsr_internal.h — shared declarations of the CUDA path (NOT shared with oracle/).
// Spec references: DESIGN.md §3 (written spec), §5 (device layout), §6 (kernels).
#pragma once
#include <cuda_runtime.h>
#include <stddef.h>
#include <stdint.h>

#include "gsr.h"

namespace gsr {

constexpr int kTile = GSR_TILE;

constexpr int kTilePix = kTile * kTile;  // 256 threads per compositing CTA, one per pixel
constexpr int kMaxC = 4096;              // clusters (mask table lives in shared memory)

// ---- device scene: SoA of 16-byte words so that every warp load is 512 B contiguous
struct DeviceScene {
  int32_t C, N, K, R, sh_degree;
  int32_t affine_cov;  // != 0: Sigma_t = L Sigma L^T with L = the 3x3 part of A_c(t) (reading I4)
  int32_t V;      // projected records per Gaussian: 2 (no position residual levels) or 4 (delta2 / delta3 given)
  int32_t n_sh4;  // float4 words of SH coefficients per Gaussian = ceil(3K/4)
  int32_t n_qw;   // 32-bit words of int8 motion coefficients per Gaussian = ceil(3R/4)
  int32_t has_delta2, has_delta3;  // the scene was given delta2 / delta3 (a missing one is stored as zeros)
  float4* g0;     // [N] mean.xyz, opacity
  float4* g1;     // [N] Sxx Sxy Sxz, tau
  float4* g2;     // [N] Syy Syz Szz, bits(cluster<<2 | level)
  float4* sh_base;  // [n_sh4][N]  flat coefficient index j*3+ch, zero padded
  float4* sh_res;   // [n_sh4][N]
  uint32_t* qw;     // [n_qw][N]   int8 q_{i,r,k} at byte (r*3+k)
  float* A0;        // [C,12]
  float* A1;        // [C,12]
  float* mscale;    // [C]
  float* delta;     // [6][N] delta2.xyz, delta3.xyz (V == 4 only), else nullptr
  float4* g1v;      // [4][N] per-depth (Sxx Sxy Sxz, tau) of scenes with attribute refinements, else nullptr
  float4* g2v;      // [4][N] per-depth (Syy Syz Szz, -)
  float* opv;       // [4][N] per-depth opacity
  float4* d_sh;     // [3][n_sh4][N] per-level colour residuals (layout of sh_base), else nullptr
  int32_t* group_off;  // [4C+1]
  float4* raw_quat;    // [N] the quaternion as given (w, x, y, z): the backward of the activation (k_project_backward.cu)
  float4* raw_ls;      // [N] log_scale.xyz, opacity_logit
  float4* raw_quat_v;  // [4][N] the raw quaternion per delivered depth (base + residuals of levels 1..v), else nullptr
  float4* raw_ls_v;    // [4][N] log_scale.xyz, opacity_logit per delivered depth, else nullptr
  float bg[3];
};

// ---- per-call constants passed by value to the kernels
struct FrameParams {
  float R[9], t[3];
  float fx, fy, cx, cy;
  int32_t W, H, TX, TY;
  float znear;
  float time;
  float basis[GSR_MAX_R];  // b_r(t) = cos(pi r t), r = 1..R, double -> fp32 on the host
  float cam_centre[3];     // -R^T t, double -> fp32 on the host
  float bg[3];
};

// ---- workspace
struct WsHeader {
  int32_t status;        // GSR_OK / GSR_E_INVALID_LEVEL / GSR_E_WORKSPACE_TOO_SMALL (latched by kernels)
  int32_t B, C, N;
  int32_t W, H, TX, TY;
  unsigned long long total_keys;  // keys the frame produced (before clamping to capacity)
  unsigned long long n_keys;      // keys actually sorted (0 if over capacity)
  long long key_capacity;
  int32_t pad[16];
};

struct Workspace {
  WsHeader* hdr;
  int8_t* depth;          // [B+1,C] validated copy of levels; row B = the full state (all 3)
  float4 *r0, *r1, *rc0, *rc1;  // [2N] projected records
  int32_t* radius;        // [2N]
  uint2* rect;            // [2N] 4 x u16: tx0,ty0,tx1,ty1
  uint32_t* depth_bits;   // [2N]
  uint32_t* count;        // [2N]
  unsigned long long* keys[2];  // [cap] [0]: sorted (tile<<32 | depth bits); [1]: per-tile segments of (depth bits<<32 | record id) before the sort
  uint32_t* vals[2];            // [cap] [0]: record ids of the sorted list; [1]: the render list (tile_render_lists in k_tile_sort)
  uint32_t* tile_cursor;  // [tiles] keys per tile, then the write cursor of the tile's segment (k_sort.cu)
  uint2* tile_range;      // [tiles] start,end into the sorted list
  uint2* render_range;    // [tiles] start,end into the render list (vals[1]): the tile's records whose q <= tau
                          // box touches a pixel of the tile, in list order (tile_render_lists in k_tile_sort)
  long long* state_counts;  // [B]
  double* sse_blk;        // [B * tiles * 8] per-(state,tile,8x4 block) squared-error partials (fused distortion)
  float4* rec;            // [4 * 2N] packed 64-byte records for the quadrant compositor (written by k_project)
  uint2* qlist;           // [4 * cap] per-(tile, quadrant) render lists of {record id, meta} (tile_render_lists in k_tile_sort)
  uint2* qrange;          // [tiles * 4] start, end into qlist
  uint32_t* uorder;       // [tiles * B] states sorted by their tile-restricted signature (k_tile_dedup)
  uint32_t* upos;         // [tiles * B] upos[tile*B + u] = index in uorder of the first member of class u
  uint32_t* n_unique;     // [tiles] number of distinct signatures
  uint32_t* work_counter; // next work item of the persistent compositing warps
  size_t bytes;           // total
};

// Which of the eight 8x4 pixel blocks of tile (tx, ty) the conservative q <= tau box of a record touches
// (DESIGN.md §4.6): centre (mx, my), half-extents (hx, hy) from k_project.  Bit k = block (k & 1, k >> 1).
// ONE definition, used by the compositor's staging and by the tile dedup (a record with mask 0 contributes
// to no pixel of the tile in any state, so it must not split signature classes either).
__device__ __forceinline__ uint32_t record_block_mask(float mx, float my, float hx, float hy, int tx, int ty) {
  const float xlo = mx - hx, xhi = mx + hx, ylo = my - hy, yhi = my + hy;
  const float X0 = (float)(tx * kTile) + 0.5f, Y0 = (float)(ty * kTile) + 0.5f;
  uint32_t ox = 0, oy = 0, m = 0;
#pragma unroll
  for (int k = 0; k < 2; ++k) ox |= (uint32_t)(xlo <= X0 + 8.0f * k + 7.0f && xhi >= X0 + 8.0f * k) << k;
#pragma unroll
  for (int k = 0; k < 4; ++k) oy |= (uint32_t)(ylo <= Y0 + 4.0f * k + 3.0f && yhi >= Y0 + 4.0f * k) << k;
#pragma unroll
  for (int k = 0; k < 8; ++k) m |= (((ox >> (k & 1)) & (oy >> (k >> 1))) & 1u) << k;
  return m;
}

// Tighter version, evaluated once per frame per (tile, record) by tile_render_lists (k_sort.cu): a block that passes the
// box test is kept only if the MINIMUM of the quadratic form q over the block's rectangle of pixel centres can
// pass the cut.  q is convex, so when the centre lies outside the rectangle the minimum sits on one of the four
// edges, where q is a 1-D quadratic (closed-form minimiser, clamped to the edge).  The block is dropped iff
// q_min > (max(tau, 0) + 0.01) (1 + m)^2 with the same m = min(1, 8e-6 kappa + 1e-3) as the box (DESIGN.md §4.6:
// fp32 evaluation of q, here and in the compositor, is within ~3e-6 kappa relative); ill-conditioned forms
// (kappa > 1e4) keep the box result.  (A, B, Cq) = (conic_a / 2, conic_b, conic_c / 2): q = (A dx + B dy) dx + Cq dy^2.
__device__ __forceinline__ uint32_t record_block_mask_tight(float mx, float my, float A, float B, float Cq, float tau,
                                                            float hx, float hy, int tx, int ty) {
  uint32_t m = record_block_mask(mx, my, hx, hy, tx, ty);
  const float det4 = 4.0f * A * Cq - B * B;  // 4 det(conic) > 0
  if (m == 0u || !(det4 > 0.0f)) return m;
  const float kappa = 4.0f * A * Cq / det4;
  if (!(kappa <= 1e4f)) return m;
  const float mm = 1.0f + fminf(1.0f, 8e-6f * kappa + 1e-3f);
  const float thr = (fmaxf(tau, 0.0f) + 1e-2f) * mm * mm;
  const float X0 = (float)(tx * kTile) + 0.5f, Y0 = (float)(ty * kTile) + 0.5f;
  const float iA = 0.5f / A, iC = 0.5f / Cq;
#pragma unroll
  for (int k = 0; k < 8; ++k) {
    if (!((m >> k) & 1u)) continue;
    const float bx = X0 + 8.0f * (k & 1), by = Y0 + 4.0f * (k >> 1);
    // d = centre - pixel; over the block dx in [dx0, dx1], dy in [dy0, dy1]
    const float dx0 = mx - (bx + 7.0f), dx1 = mx - bx, dy0 = my - (by + 3.0f), dy1 = my - by;
    if (dx0 <= 0.0f && dx1 >= 0.0f && dy0 <= 0.0f && dy1 >= 0.0f) continue;  // centre inside: q_min = 0
    float qmin = 3.4e38f;
#pragma unroll
    for (int e = 0; e < 2; ++e) {
      const float dx = e ? dx1 : dx0;                       // vertical edges: dx fixed, dy free
      float dy = fminf(dy1, fmaxf(dy0, -(B * dx) * iC));
      qmin = fminf(qmin, (A * dx + B * dy) * dx + Cq * dy * dy);
      const float dyf = e ? dy1 : dy0;                      // horizontal edges: dy fixed, dx free
      float dxs = fminf(dx1, fmaxf(dx0, -(B * dyf) * iA));
      qmin = fminf(qmin, (A * dxs + B * dyf) * dxs + Cq * dyf * dyf);
    }
    if (qmin > thr) m &= ~(1u << k);
  }
  return m;
}


size_t carve_workspace(Workspace* ws, void* base, int32_t N, int32_t C, int32_t B, int32_t tiles, long long cap);
long long default_key_capacity(int32_t N);
// carve_workspace / default_key_capacity take HALF the number of projected records (= N when V == 2)
inline int32_t rec_half(const DeviceScene& d) { return (int32_t)((long long)d.N * d.V / 2); }

// ---- kernel launchers (each only enqueues on `st`)
void launch_init_header(Workspace& ws, int32_t B, int32_t C, int32_t N, const FrameParams& fp, long long cap,
                        cudaStream_t st);
void launch_validate_levels(const int8_t* levels, int32_t B, int32_t C, Workspace& ws, cudaStream_t st);
void launch_project(const DeviceScene& sc, const FrameParams& fp, Workspace& ws, cudaStream_t st);
void launch_bin_and_sort(const DeviceScene& sc, const FrameParams& fp, Workspace& ws, long long cap, cudaStream_t st);
void launch_state_counts(const DeviceScene& sc, Workspace& ws, int32_t B, cudaStream_t st);
// composites B states whose depth rows start at `depth_rows` (ws.depth, or ws.depth + B*C for the full state)
void launch_composite(const DeviceScene& sc, const FrameParams& fp, Workspace& ws, const int8_t* depth_rows,
                      int32_t B, float* out, const float* ref, double* mse, float* psnr, cudaStream_t st);
// instrumented run of the same kernel: counts[0] = (pixel, record) pairs evaluated with >= 1 live present
// state, counts[1] = (pixel, record, state) updates on live present states, counts[2] = logical pairs E
void launch_composite_count(const DeviceScene& sc, const FrameParams& fp, Workspace& ws, const int8_t* depth_rows,
                            int32_t B, unsigned long long* counts, cudaStream_t st);
void count_launches(int n);
struct CompositeArgs;
void launch_composite_q(const CompositeArgs& a, int S, bool count, cudaStream_t st);
// backward of a4 (k_backward.cu): grad [records, 12], zeroed by the call
void launch_objective_weights(const double* d, int32_t n, double w_mean, double w_cvar, double alpha,
                              const int32_t* prev, const int32_t* next, int32_t n_pairs, double w_mono, double* w,
                              cudaStream_t st);
void launch_flicker_backward(const float* a1, const float* a2, const float* r1, const float* r2, int32_t B, int32_t H,
                             int32_t W, const double* weight, float* g1, float* g2, cudaStream_t st);
constexpr long long kStaticPartials = 1ll << 20;  // doubles of file-scope scratch behind gsr_distortion_static (8 MiB)
int launch_distortion_static(const float* imgs, const float* ref, int32_t B, int32_t H, int32_t W, double* mse,
                             float* psnr, cudaStream_t st);
int launch_distortion_backward(const float* imgs, const float* ref, int32_t B, int32_t H, int32_t W,
                               const double* weight, double lambda, float* out, double* ref_planes, cudaStream_t st);
void launch_project_backward(const DeviceScene& sc, const FrameParams& fp, const float* grad_rec, float* g_gauss,
                             float* g_shb, float* g_shr, float* g_cluster, cudaStream_t st);
void launch_project_backward4(const DeviceScene& sc, const FrameParams& fp, const float* grad_rec, float* g_gauss,
                              float* g_shb, float* g_shr, float* g_cluster, float* g_delta, float* g_attr, float* g_dsh,
                              cudaStream_t st);
void launch_backward(const DeviceScene& sc, const WsHeader& h, Workspace& ws, const float* images, const float* gimg,
                     float* grad, cudaStream_t st);
void launch_distortion_finalize_blk(const double* blk, int32_t B, int32_t tiles, int64_t n_values, double* mse,
                                    float* psnr, cudaStream_t st);
bool launch_tile_dedup(const DeviceScene& sc, const FrameParams& fp, Workspace& ws, const int8_t* depth_rows,
                       int32_t B, cudaStream_t st);
void launch_distortion(const float* imgs, const float* ref, int32_t B, int32_t H, int32_t W, double* part,
                       double* mse, float* psnr, cudaStream_t st);
void launch_distortion_finalize(const double* part, int32_t B, int32_t tiles, int64_t n_values, double* mse,
                                float* psnr, cudaStream_t st);
// B = number of states behind mse / psnr (range of the pair indices), or < 0 if the caller did not say
void launch_group_utility(const double* mse, const float* psnr, int32_t B, const int32_t* iwo, const int32_t* iw,
                          const int32_t* gid, int32_t n_pairs, int32_t G, gsr_utility* out, double* dmse,
                          double* ddb, cudaStream_t st);
void launch_close_levels(const uint8_t* mask, int64_t n, int8_t* depth, uint8_t* closure, cudaStream_t st);
void launch_filter_keys(const DeviceScene& sc, Workspace& ws, int32_t b, uint32_t* tile, uint32_t* dbits,
                        int32_t* gi, unsigned long long* n_out, long long cap, cudaStream_t st);

// scheduling frontier / atlas (k_policy.cu)
void launch_wire_bytes(const long long* raw, int32_t C, long long* wire, cudaStream_t st);
void launch_frontier_order(const double* score, const long long* wire, int32_t C, int32_t policy, int32_t* order,
                           long long* cum, cudaStream_t st);
void launch_frontier_states(const int32_t* order, const long long* wire, int32_t C, const long long* budgets,
                            int32_t nb, int8_t* levels, long long* used, int32_t* n_groups, cudaStream_t st);
void launch_state_bytes(const int8_t* levels, int32_t B, int32_t C, const long long* wire, long long* out,
                        cudaStream_t st);
void launch_best_under_budget(const float* psnr, const long long* bytes, int32_t B, const long long* budgets,
                              int32_t nb, int32_t* best, cudaStream_t st);

// richer distortion / risk reductions (k_metrics.cu)
void launch_ssim(const float* imgs, const float* ref, int32_t B, int32_t H, int32_t W, const double* mse, double* part,
                 double* ssim, double* dmix, cudaStream_t st);
void launch_flicker(const float* a1, const float* a2, const float* r1, const float* r2, int32_t B, int32_t H, int32_t W,
                    double* part, double* out, cudaStream_t st);
void launch_risk_reduce(const void* values, int32_t is_f32, int32_t n, double alpha, int32_t upper, gsr_risk* out,
                        cudaStream_t st);
// n = length of d (range of the indices), or < 0 if the caller did not say
void launch_prefix_monotonicity(const double* d, int32_t n, const int32_t* prev, const int32_t* next, int32_t n_pairs,
                                double* m_out, int32_t* viol, cudaStream_t st);

// delivery-mask sampler (k_delivery.cu)
size_t delivery_workspace_bytes(int32_t C);
void launch_sample_delivery(const long long* raw, const int32_t* order, int32_t C, const gsr_loss_model& m,
                            const int32_t* budget, int32_t W, int32_t world0, uint8_t* mask, int8_t* levels,
                            long long* pk_start, cudaStream_t st);

void set_error(const char* fmt, ...);

// Index arrays handed to the device-pointer calls (send orders, pair lists, prefix pairs) are checked IN the
// kernels: an entry out of range is skipped and its bit is OR-ed into a per-device error word that
// gsr_index_status reads and clears.  Returns nullptr if the word cannot be allocated.
enum : int { kBadOrder = 1, kBadPairIndex = 2, kBadGroupId = 4, kBadPrefixIndex = 8 };
int* device_error_word();

}  // namespace gsr
