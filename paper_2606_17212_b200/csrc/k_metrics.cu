// k_metrics.cu — richer distortion and risk reductions:
//   SSIM and D = MSE + 0.20 (1 - SSIM)        PAPER.md:72   (reading G1)
//   mean / CVaR / quantile / worst over states PAPER.md:68-76 (reading G2)
//   temporal flicker F                          PAPER.md:70   (reading G3)
//   prefix monotonicity M                       PAPER.md:70   (reading G4)
// SSIM and flicker read materialised images ([B,H,W,3] fp32) and are reduced with the canonical tree of
// reduce.cuh (warp butterfly in double, warps in index order, tiles in index order), so they are
// deterministic.  The reductions over states are single-CTA, latency-bound helpers.
#include "gsr_internal.h"
#include "reduce.cuh"

namespace gsr {

constexpr int kSsimR = 5;                      // window radius (11 x 11)
constexpr double kSsimC1 = 0.01 * 0.01, kSsimC2 = 0.03 * 0.03;

struct SsimWindow { double g[2 * kSsimR + 1]; };  // normalised weights, evaluated on the host

// One CTA = one 32x32 block of pixels (2 x 2 tiles) of one state.  Per channel: stage the 42x42 halo of img and ref
// (zero outside the image: reading G1's zero padding; converted to double once), blur the five moments x, y, xx, yy,
// xy horizontally into 42 rows x 32 columns, then vertically.  Every blur step gives a thread a run of 4 consecutive
// outputs along the blur direction, so that the 14 inputs are read once into registers instead of 11 loads per output
// (the first version of this kernel, one thread per pixel of a 16x16 tile, was bound by the shared-memory
// instruction queue and the float -> double conversions, like the first k_distortion_backward: 7.3 ms for
// 128 x 800 x 800, now 4.4 ms).  The moments are accumulated in DOUBLE: the variance terms E[x^2] - mu^2
// cancel against C2 = 9e-4, and fp32 moments leave a systematic 4e-5 error on flat regions (measured).
// Partials: one double per (state, 16x16 tile) as before (k_ssim_finalize is unchanged); within a tile the 64 run
// sums are added by one warp with the butterfly: deterministic.
constexpr int kSsimT = 32;                        // block edge
constexpr int kSsimIn = kSsimT + 2 * kSsimR;      // 42
constexpr int kSsimThreads = 384;
constexpr int kSsimRun = 4;

struct SsimSmem {
  double x[kSsimIn][kSsimIn + 1], y[kSsimIn][kSsimIn + 1];
  double h[5][kSsimIn][kSsimT + 1];
  double run[(kSsimT / kSsimRun) * kSsimT];  // [row group][column]: sum of the SSIM map over the run's 4 pixels, 3 channels
};

__global__ void __launch_bounds__(kSsimThreads, 2) k_ssim_blocks(const float* __restrict__ imgs,
                                                                const float* __restrict__ ref, int W, int H, int TXB,
                                                                int TX, int TY, int tiles, SsimWindow win,
                                                                double* __restrict__ part) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  SsimSmem& s = *reinterpret_cast<SsimSmem*>(smem_raw);
  const int tid = threadIdx.x;
  const int blk = blockIdx.x, b = blockIdx.y;
  const int bx = blk % TXB, by = blk / TXB;
  const int x0 = bx * kSsimT, y0 = by * kSsimT;
  const float* img = imgs + (size_t)b * H * W * 3;
  constexpr int kItemsE = (kSsimT / kSsimRun) * kSsimT;  // 256 runs of the vertical step
  double acc = 0.0;  // the thread's run (tid < 256) over the three channels
  for (int ch = 0; ch < 3; ++ch) {
    for (int i = tid; i < kSsimIn * kSsimIn; i += kSsimThreads) {
      const int hy = i / kSsimIn, hx = i - hy * kSsimIn;
      const int gx = x0 + hx - kSsimR, gy = y0 + hy - kSsimR;
      float vx = 0.0f, vy = 0.0f;
      if (gx >= 0 && gx < W && gy >= 0 && gy < H) {
        const size_t p = ((size_t)gy * W + gx) * 3 + ch;
        vx = __ldg(img + p);
        vy = __ldg(ref + p);
      }
      s.x[hy][hx] = (double)vx;
      s.y[hy][hx] = (double)vy;
    }
    __syncthreads();
    // horizontal: 42 rows x 8 runs of 4 columns; lanes run over rows
    for (int i = tid; i < kSsimIn * (kSsimT / kSsimRun); i += kSsimThreads) {
      const int grp = i / kSsimIn, r = i - grp * kSsimIn, c0 = grp * kSsimRun;
      double xv[kSsimRun + 2 * kSsimR], yv[kSsimRun + 2 * kSsimR];
#pragma unroll
      for (int j = 0; j < kSsimRun + 2 * kSsimR; ++j) { xv[j] = s.x[r][c0 + j]; yv[j] = s.y[r][c0 + j]; }
#pragma unroll
      for (int o = 0; o < kSsimRun; ++o) {
        double m0 = 0., m1 = 0., m2 = 0., m3 = 0., m4 = 0.;
#pragma unroll
        for (int k = 0; k <= 2 * kSsimR; ++k) {
          const double a = xv[o + k], c = yv[o + k], g = win.g[k];
          m0 = fma(g, a, m0);
          m1 = fma(g, c, m1);
          m2 = fma(g, a * a, m2);
          m3 = fma(g, c * c, m3);
          m4 = fma(g, a * c, m4);
        }
        s.h[0][r][c0 + o] = m0; s.h[1][r][c0 + o] = m1; s.h[2][r][c0 + o] = m2; s.h[3][r][c0 + o] = m3; s.h[4][r][c0 + o] = m4;
      }
    }
    __syncthreads();
    // vertical: 32 columns x 8 runs of 4 rows; lanes run over columns; then the SSIM map of the run's pixels
    if (tid < kItemsE) {
      const int grp = tid / kSsimT, c = tid - grp * kSsimT, r0 = grp * kSsimRun;
      double mo[5][kSsimRun];
#pragma unroll
      for (int m = 0; m < 5; ++m) {
        double v[kSsimRun + 2 * kSsimR];
#pragma unroll
        for (int j = 0; j < kSsimRun + 2 * kSsimR; ++j) v[j] = s.h[m][r0 + j][c];
#pragma unroll
        for (int o = 0; o < kSsimRun; ++o) {
          double t = 0.;
#pragma unroll
          for (int k = 0; k <= 2 * kSsimR; ++k) t = fma(win.g[k], v[o + k], t);
          mo[m][o] = t;
        }
      }
      const int px = x0 + c;
#pragma unroll
      for (int o = 0; o < kSsimRun; ++o) {
        const int py = y0 + r0 + o;
        const double mx = mo[0][o], my = mo[1][o];
        const double sxx = mo[2][o] - mx * mx, syy = mo[3][o] - my * my, sxy = mo[4][o] - mx * my;
        const double num = (2.0 * mx * my + kSsimC1) * (2.0 * sxy + kSsimC2);
        const double den = (mx * mx + my * my + kSsimC1) * (sxx + syy + kSsimC2);
        if (px < W && py < H) acc += num / den;
      }
    }
    __syncthreads();
  }
  if (tid < kItemsE) s.run[tid] = acc;
  __syncthreads();
  // the four 16x16 tiles of the block: tile (tcx, tcy) owns the runs with column / 16 == tcx and row group / 4 == tcy
  const int w = tid >> 5, lane = tid & 31;
  if (w < 4) {
    const int tcx = w & 1, tcy = w >> 1;
    // 64 runs: 4 row groups x 16 columns; lane takes two of them in a fixed order
    const int g0 = 4 * tcy + (lane >> 4), cc = 16 * tcx + (lane & 15);
    const double v = s.run[g0 * kSsimT + cc] + s.run[(g0 + 2) * kSsimT + cc];
    const double t = warp_sum_butterfly(v);
    const int tx16 = 2 * bx + tcx, ty16 = 2 * by + tcy;
    if (lane == 0 && tx16 < TX && ty16 < TY) part[(size_t)b * tiles + (size_t)ty16 * TX + tx16] = t;
  }
}

// one warp per state: tiles in index order (lane-strided), then the butterfly; SSIM and the mixed distortion
__global__ void __launch_bounds__(128) k_ssim_finalize(const double* __restrict__ part, int B, int tiles, double inv_n,
                                                       const double* __restrict__ mse, double* __restrict__ ssim,
                                                       double* __restrict__ dmix) {
  const int b = blockIdx.x * 4 + (threadIdx.x >> 5), lane = threadIdx.x & 31;
  if (b >= B) return;
  double acc = 0.0;
  for (int k = lane; k < tiles; k += 32) acc += part[(size_t)b * tiles + k];
  acc = warp_sum_butterfly(acc);
  if (lane == 0) {
    const double s = acc * inv_n;
    if (ssim) ssim[b] = s;
    if (dmix && mse) dmix[b] = mse[b] + 0.20 * (1.0 - s);
  }
}

// ---- flicker (reading G3): same pixel->thread mapping and tree as gsr_distortion
__global__ void __launch_bounds__(kTilePix) k_flicker_tiles(const float* __restrict__ a1, const float* __restrict__ a2,
                                                            const float* __restrict__ r1, const float* __restrict__ r2,
                                                            int W, int H, int TX, int tiles, double* __restrict__ part) {
  __shared__ double s_red[8];
  const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
  const int tile = blockIdx.x, b = blockIdx.y;
  const int x = (tile % TX) * kTile + 8 * (w & 1) + (lane & 7), y = (tile / TX) * kTile + 4 * (w >> 1) + (lane >> 3);
  float e = 0.0f;
  if (x < W && y < H) {
    const size_t p = ((size_t)y * W + x) * 3;
    const size_t o = (size_t)b * H * W * 3 + p;
    float d[3];
#pragma unroll
    for (int ch = 0; ch < 3; ++ch)
      d[ch] = __fsub_rn(__fsub_rn(a2[o + ch], a1[o + ch]), __fsub_rn(__ldg(r2 + p + ch), __ldg(r1 + p + ch)));
    e = __fmaf_rn(d[2], d[2], __fmaf_rn(d[1], d[1], __fmul_rn(d[0], d[0])));
  }
  const double ws = warp_sum_butterfly((double)e);
  if (lane == 0) s_red[w] = ws;
  __syncthreads();
  if (tid == 0) {
    double acc = s_red[0];
#pragma unroll
    for (int k = 1; k < 8; ++k) acc += s_red[k];
    part[(size_t)b * tiles + tile] = acc;
  }
}

// ---- reductions over states (reading G2): one CTA, any n; order statistics by exact MSB-first radix select
constexpr int kRiskThreads = 256;

__device__ __forceinline__ unsigned long long risk_key(double v) {
  unsigned long long u = (unsigned long long)__double_as_longlong(v);
  return (u & 0x8000000000000000ull) ? ~u : (u | 0x8000000000000000ull);
}
__device__ __forceinline__ double risk_unkey(unsigned long long k) {
  unsigned long long u = (k & 0x8000000000000000ull) ? (k & 0x7FFFFFFFFFFFFFFFull) : ~k;
  return __longlong_as_double((long long)u);
}
__device__ __forceinline__ double risk_load(const void* v, int is_f32, int i) {
  return is_f32 ? (double)((const float*)v)[i] : ((const double*)v)[i];
}

template <typename T>
__device__ __forceinline__ T risk_block_sum(T v, T* sm) {
  sm[threadIdx.x] = v;
  __syncthreads();
  for (int k = kRiskThreads / 2; k > 0; k >>= 1) {
    if (threadIdx.x < k) sm[threadIdx.x] += sm[threadIdx.x + k];
    __syncthreads();
  }
  T r = sm[0];
  __syncthreads();
  return r;
}

// k-th smallest (0-based) value
__device__ double risk_select(const void* v, int is_f32, int n, int k, unsigned long long* sm) {
  unsigned long long ans = 0ull;
  for (int bit = 63; bit >= 0; --bit) {
    const unsigned long long cand = ans | (1ull << bit);
    unsigned long long c = 0;
    for (int i = threadIdx.x; i < n; i += kRiskThreads) c += risk_key(risk_load(v, is_f32, i)) < cand;
    c = risk_block_sum<unsigned long long>(c, sm);
    if (c <= (unsigned long long)k) ans = cand;  // at most k keys below cand => the k-th key is >= cand
  }
  return risk_unkey(ans);
}

__global__ void __launch_bounds__(kRiskThreads) k_risk_reduce(const void* __restrict__ v, int is_f32, int n, double alpha,
                                                              int upper, gsr_risk* __restrict__ out) {
  __shared__ double sm_d[kRiskThreads];
  __shared__ unsigned long long sm_c[kRiskThreads];
  gsr_risk r;
  r.mean = r.cvar = r.quantile = r.worst = 0.0;
  r.count = (double)n;
  if (n > 0) {
    double s = 0.0;
    for (int i = threadIdx.x; i < n; i += kRiskThreads) s += risk_load(v, is_f32, i);
    r.mean = risk_block_sum<double>(s, sm_d) / (double)n;
    int k = (int)ceil(alpha * (double)n);
    k = k < 1 ? 1 : (k > n ? n : k);
    // threshold = the mildest of the k worst values; the tail sum takes everything strictly worse plus the
    // right number of copies of the threshold (ties)
    const double thr = risk_select(v, is_f32, n, upper ? n - k : k - 1, sm_c);
    double ts = 0.0;
    unsigned long long tc = 0;
    for (int i = threadIdx.x; i < n; i += kRiskThreads) {
      const double x = risk_load(v, is_f32, i);
      if (upper ? x > thr : x < thr) { ts += x; ++tc; }
    }
    ts = risk_block_sum<double>(ts, sm_d);
    tc = risk_block_sum<unsigned long long>(tc, sm_c);
    r.cvar = (ts + (double)(k - (int)tc) * thr) / (double)k;
    const double pos = (upper ? 1.0 - alpha : alpha) * (double)(n - 1);
    const int lo = (int)floor(pos);
    const int hi = lo + 1 < n ? lo + 1 : n - 1;
    const double vlo = risk_select(v, is_f32, n, lo, sm_c);
    const double vhi = hi == lo ? vlo : risk_select(v, is_f32, n, hi, sm_c);
    r.quantile = vlo + (pos - (double)lo) * (vhi - vlo);
    r.worst = risk_select(v, is_f32, n, upper ? n - 1 : 0, sm_c);
  }
  if (threadIdx.x == 0) *out = r;
}

// ---- prefix monotonicity (reading G4)
__global__ void __launch_bounds__(kRiskThreads) k_prefix_monotonicity(const double* __restrict__ d, int n,
                                                                      const int* __restrict__ prev,
                                                                      const int* __restrict__ next, int n_pairs,
                                                                      double* __restrict__ m_out, int* __restrict__ viol,
                                                                      int* __restrict__ err) {
  __shared__ double sm_d[kRiskThreads];
  __shared__ unsigned long long sm_c[kRiskThreads];
  double s = 0.0;
  unsigned long long c = 0;
  for (int p = threadIdx.x; p < n_pairs; p += kRiskThreads) {
    const int a = prev[p], b = next[p];
    if (a < 0 || b < 0 || (n >= 0 && (a >= n || b >= n))) {  // refused pair: contributes nothing, the caller is told
      if (err) atomicOr(err, kBadPrefixIndex);
      continue;
    }
    const double inc = d[b] - d[a];
    if (inc > 0.0) { s += inc; ++c; }
  }
  s = risk_block_sum<double>(s, sm_d);
  c = risk_block_sum<unsigned long long>(c, sm_c);
  if (threadIdx.x == 0) {
    if (m_out) *m_out = s;
    if (viol) *viol = (int)c;
  }
}

// ---- dL/dD_b of L = w_mean mean(D) + w_cvar CVaR_alpha(D) + w_mono M(D) (Eq. (2)):
//      1/n each; 1/k for every value strictly above the CVaR threshold and the remaining (k - #above)/k shared
//      equally by the values equal to it (a subgradient, reading L1); +w_mono on next, -w_mono on prev of every
//      violated pair.  One CTA.
__global__ void __launch_bounds__(kRiskThreads) k_objective_weights(const double* __restrict__ d, int n, double w_mean,
                                                                    double w_cvar, double alpha,
                                                                    const int* __restrict__ prev,
                                                                    const int* __restrict__ next, int n_pairs,
                                                                    double w_mono, double* __restrict__ w,
                                                                    int* __restrict__ err) {
  __shared__ unsigned long long sm_c[kRiskThreads];
  if (n <= 0) return;
  int k = (int)ceil(alpha * (double)n);
  k = k < 1 ? 1 : (k > n ? n : k);
  const double thr = risk_select(d, 0, n, n - k, sm_c);
  unsigned long long above = 0, ties = 0;
  for (int i = threadIdx.x; i < n; i += kRiskThreads) {
    above += d[i] > thr;
    ties += d[i] == thr;
  }
  above = risk_block_sum<unsigned long long>(above, sm_c);
  ties = risk_block_sum<unsigned long long>(ties, sm_c);
  const double share = ties ? w_cvar * (double)(k - (int)above) / ((double)ties * (double)k) : 0.0;
  for (int i = threadIdx.x; i < n; i += kRiskThreads)
    w[i] = w_mean / (double)n + (d[i] > thr ? w_cvar / (double)k : (d[i] == thr ? share : 0.0));
  __syncthreads();
  for (int p = threadIdx.x; p < n_pairs; p += kRiskThreads) {
    const int a = prev[p], b = next[p];
    if (a < 0 || b < 0 || a >= n || b >= n) {
      if (err) atomicOr(err, kBadPrefixIndex);
      continue;
    }
    if (d[b] - d[a] > 0.0) {
      atomicAdd(w + b, w_mono);
      atomicAdd(w + a, -w_mono);
    }
  }
}

// ---- d/d(imgs_t1), d/d(imgs_t2) of sum_b weight_b F_b (reading G3): the forward's fp32 differences, then 2 e / (3 H W)
__global__ void k_flicker_backward(const float* __restrict__ a1, const float* __restrict__ a2, const float* __restrict__ r1,
                                   const float* __restrict__ r2, size_t img, const double* __restrict__ weight,
                                   float* __restrict__ g1, float* __restrict__ g2) {
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int b = blockIdx.y;
  if (i >= img) return;
  const size_t o = (size_t)b * img + i;
  const float e = __fsub_rn(__fsub_rn(a2[o], a1[o]), __fsub_rn(__ldg(r2 + i), __ldg(r1 + i)));
  const double g = (weight ? weight[b] : 1.0) * 2.0 * (double)e / (double)img;
  if (g2) g2[o] = (float)g;
  if (g1) g1[o] = (float)(-g);
}

// ------------------------------------------------------------------------------------------------ launchers
void launch_ssim(const float* imgs, const float* ref, int32_t B, int32_t H, int32_t W, const double* mse, double* part,
                 double* ssim, double* dmix, cudaStream_t st) {
  if (B == 0) return;
  const int TX = (W + kTile - 1) / kTile, TY = (H + kTile - 1) / kTile, tiles = TX * TY;
  SsimWindow win;
  double g[2 * kSsimR + 1], sum = 0.0;
  for (int k = 0; k <= 2 * kSsimR; ++k) {  // exp(-(k-5)^2 / (2 * 1.5^2)), normalised
    g[k] = exp(-(double)((k - kSsimR) * (k - kSsimR)) / (2.0 * 1.5 * 1.5));
    sum += g[k];
  }
  for (int k = 0; k <= 2 * kSsimR; ++k) win.g[k] = g[k] / sum;
  const int TXB = (W + kSsimT - 1) / kSsimT, TYB = (H + kSsimT - 1) / kSsimT;
  // 84 KB of shared memory per CTA: opt in (per device, cheap: on every call)
  cudaFuncSetAttribute(k_ssim_blocks, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(SsimSmem));
  for (int b0 = 0; b0 < B; b0 += 65535) {  // gridDim.y limit
    const int nb = B - b0 < 65535 ? B - b0 : 65535;
    k_ssim_blocks<<<dim3(TXB * TYB, nb), kSsimThreads, sizeof(SsimSmem), st>>>(
        imgs + (size_t)b0 * H * W * 3, ref, W, H, TXB, TX, TY, tiles, win, part + (size_t)b0 * tiles);
    count_launches(1);
  }
  k_ssim_finalize<<<(B + 3) / 4, 128, 0, st>>>(part, B, tiles, 1.0 / (3.0 * (double)W * (double)H), mse, ssim, dmix);
  count_launches(1);
}

void launch_flicker(const float* a1, const float* a2, const float* r1, const float* r2, int32_t B, int32_t H, int32_t W,
                    double* part, double* out, cudaStream_t st) {
  if (B == 0) return;
  const int TX = (W + kTile - 1) / kTile, TY = (H + kTile - 1) / kTile, tiles = TX * TY;
  for (int b0 = 0; b0 < B; b0 += 65535) {
    const int nb = B - b0 < 65535 ? B - b0 : 65535;
    const size_t off = (size_t)b0 * H * W * 3;
    k_flicker_tiles<<<dim3(tiles, nb), kTilePix, 0, st>>>(a1 + off, a2 + off, r1, r2, W, H, TX, tiles,
                                                         part + (size_t)b0 * tiles);
    count_launches(1);
  }
  launch_distortion_finalize(part, B, tiles, (int64_t)3 * W * H, out, nullptr, st);
}

void launch_risk_reduce(const void* values, int32_t is_f32, int32_t n, double alpha, int32_t upper, gsr_risk* out,
                        cudaStream_t st) {
  k_risk_reduce<<<1, kRiskThreads, 0, st>>>(values, is_f32, n, alpha, upper, out);
  count_launches(1);
}

void launch_prefix_monotonicity(const double* d, int32_t n, const int32_t* prev, const int32_t* next, int32_t n_pairs,
                                double* m_out, int32_t* viol, cudaStream_t st) {
  k_prefix_monotonicity<<<1, kRiskThreads, 0, st>>>(d, n, prev, next, n_pairs, m_out, viol, device_error_word());
  count_launches(1);
}

void launch_objective_weights(const double* d, int32_t n, double w_mean, double w_cvar, double alpha,
                              const int32_t* prev, const int32_t* next, int32_t n_pairs, double w_mono, double* w,
                              cudaStream_t st) {
  if (n <= 0) return;
  k_objective_weights<<<1, kRiskThreads, 0, st>>>(d, n, w_mean, w_cvar, alpha, prev, next, n_pairs, w_mono, w,
                                                  device_error_word());
  count_launches(1);
}

void launch_flicker_backward(const float* a1, const float* a2, const float* r1, const float* r2, int32_t B, int32_t H,
                             int32_t W, const double* weight, float* g1, float* g2, cudaStream_t st) {
  if (B == 0) return;
  const size_t img = (size_t)H * W * 3;
  for (int b0 = 0; b0 < B; b0 += 65535) {
    const int nb = B - b0 < 65535 ? B - b0 : 65535;
    k_flicker_backward<<<dim3((unsigned)((img + 255) / 256), nb), 256, 0, st>>>(
        a1 + (size_t)b0 * img, a2 + (size_t)b0 * img, r1, r2, img, weight ? weight + b0 : nullptr,
        g1 ? g1 + (size_t)b0 * img : nullptr, g2 ? g2 + (size_t)b0 * img : nullptr);
    count_launches(1);
  }
}

}  // namespace gsr
