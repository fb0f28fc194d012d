// k_distortion_backward.cu — d/d(image) of sum_b weight_b D_b, D = MSE + lambda (1 - SSIM) (the term
// E_w[D_w] of Eq. (2) with "D = MSE + 0.20(1 - SSIM)"; SSIM per reading G1 of DESIGN.md §12).
//
// Per channel, with the 11 x 11 Gaussian window w (zero padding) and m1 = w*x, m2 = w*(x x), m12 = w*(x y):
//   ssim = N1 N2 / (D1 D2), N1 = 2 mu_x mu_y + C1, N2 = 2 s_xy + C2, D1 = mu_x^2 + mu_y^2 + C1, D2 = s_xx + s_yy + C2
//   b = d ssim/d m2  = -N1 N2 / (D1 D2^2)
//   c = d ssim/d m12 = 2 N1 / (D1 D2)
//   a = d ssim/d m1  = 2 mu_y N2 / (D1 D2) - 2 mu_x N1 N2 / (D1^2 D2) - 2 mu_x b - mu_y c
//   d mean(ssim)/dx = ( w*a + 2 x w*b + y w*c ) / (3 H W)          (the window is symmetric)
//   dL/dx = weight_b ( 2 (x - y) / (3 H W) - lambda d mean(ssim)/dx )
// One CTA per (32 x 32 block of pixels, state): the block with a halo of 10 pixels is staged, the three moments that
// depend on the image are blurred on the block-plus-5 region (42 x 42), a, b, c are formed there (zero outside the
// image: no SSIM value exists there) and blurred back onto the block.  The two moments of the reference alone
// (mu_y, w*(y y)) do not depend on the state: k_ref_moments computes them once per call into the workspace.
// Moments and maps in double, like the forward SSIM (k_metrics.cu): the variance terms cancel against C2 = 9e-4.
#include "gsr_internal.h"

namespace gsr {

constexpr int kDbR = 5;                    // window radius
constexpr int kDbT = 32;                   // block edge
constexpr int kDbIn = kDbT + 4 * kDbR;     // 52: staged pixels per side
constexpr int kDbMid = kDbT + 2 * kDbR;    // 42: positions where the SSIM map is needed
constexpr int kDbThreads = 384;
constexpr double kDbC1 = 0.01 * 0.01, kDbC2 = 0.03 * 0.03;

struct DbWindow { double g[2 * kDbR + 1]; };

struct DbSmem {
  // staging, converted once (F2F runs at a fraction of the DFMA rate); dead after step B, when a, b, c
  // ([3][kDbMid][kDbMid + 1] doubles) take its place — 106 KB in all, so that two CTAs share an SM and one computes
  // while the other waits at a barrier
  double x[kDbIn][kDbIn + 1], y[kDbIn][kDbIn + 1];
  double h[3][kDbIn][kDbMid + 1];   // x, x x, x y blurred along x; reused for the maps blurred along x: [3][kDbMid][kDbT + 1]
  float cx[kDbT][kDbT + 1], cy[kDbT][kDbT + 1];  // the block's own pixels, for step E
};
static_assert(sizeof(double) * 3 * kDbMid * (kDbMid + 1) <= sizeof(double) * 2 * kDbIn * (kDbIn + 1), "a, b, c alias the staging");

// Every blur step gives a thread a run of kRun consecutive outputs along the blur direction: the kRun + 10 inputs
// are read once into registers (a sliding window), instead of 11 loads per output — the first version of this
// kernel was bound by the shared-memory instruction queue (mio_throttle 3.5 per issue), not by the DFMAs.
constexpr int kRunB = 6, kRunD = 4;  // 42 = 7 * 6 positions per row / column of the middle region; 32 = 8 * 4 of the block

// mu_y = w*y and w*(y y) of the reference, double [H, W, 3] each (the image layout), zero padding
__global__ void __launch_bounds__(kTilePix) k_ref_moments(const float* __restrict__ ref, int W, int H, int TX,
                                                          DbWindow win, double* __restrict__ my,
                                                          double* __restrict__ eyy) {
  constexpr int kHalo = kTile + 2 * kDbR;  // 26
  __shared__ float s_y[kHalo][kHalo + 1];
  __shared__ double s_h[2][kHalo][kTile + 1];
  const int tid = threadIdx.x, tile = blockIdx.x;
  const int x0 = (tile % TX) * kTile, y0 = (tile / TX) * kTile;
  const int ty = tid / kTile, tx = tid % kTile;
  for (int ch = 0; ch < 3; ++ch) {
    for (int i = tid; i < kHalo * kHalo; i += kTilePix) {
      const int hy = i / kHalo, hx = i - hy * kHalo;
      const int qx = x0 + hx - kDbR, qy = y0 + hy - kDbR;
      s_y[hy][hx] = (qx >= 0 && qx < W && qy >= 0 && qy < H) ? __ldg(ref + ((size_t)qy * W + qx) * 3 + ch) : 0.0f;
    }
    __syncthreads();
    for (int i = tid; i < kHalo * kTile; i += kTilePix) {
      const int r = i / kTile, c = i - r * kTile;
      double a0 = 0, a1 = 0;
#pragma unroll
      for (int k = 0; k <= 2 * kDbR; ++k) {
        const double yv = (double)s_y[r][c + k], g = win.g[k];
        a0 += g * yv; a1 += g * (yv * yv);
      }
      s_h[0][r][c] = a0; s_h[1][r][c] = a1;
    }
    __syncthreads();
    if (x0 + tx < W && y0 + ty < H) {
      double a0 = 0, a1 = 0;
#pragma unroll
      for (int k = 0; k <= 2 * kDbR; ++k) {
        a0 += win.g[k] * s_h[0][ty + k][tx]; a1 += win.g[k] * s_h[1][ty + k][tx];
      }
      const size_t o = ((size_t)(y0 + ty) * W + (x0 + tx)) * 3 + ch;
      my[o] = a0;
      eyy[o] = a1;
    }
    __syncthreads();
  }
}

__global__ void __launch_bounds__(kDbThreads, 2) k_distortion_backward(const float* __restrict__ imgs,
                                                                    const float* __restrict__ ref, int W, int H, int TX,
                                                                    const double* __restrict__ ref_my,
                                                                    const double* __restrict__ ref_eyy,
                                                                    const double* __restrict__ weight, double lambda,
                                                                    DbWindow win, float* __restrict__ out) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  DbSmem& s = *reinterpret_cast<DbSmem*>(smem_raw);
  double(*gx)[kDbMid][kDbT + 1] = reinterpret_cast<double(*)[kDbMid][kDbT + 1]>(&s.h[0][0][0]);
  double(*sm)[kDbMid][kDbMid + 1] = reinterpret_cast<double(*)[kDbMid][kDbMid + 1]>(&s.x[0][0]);
  const int tid = threadIdx.x, tile = blockIdx.x, b = blockIdx.y;
  const int x0 = (tile % TX) * kDbT, y0 = (tile / TX) * kDbT;
  const size_t img = (size_t)H * W * 3;
  const float* im = imgs + (size_t)b * img;
  const double wb = weight ? weight[b] : 1.0;
  const double inv_n = 1.0 / (3.0 * (double)W * (double)H);
  for (int ch = 0; ch < 3; ++ch) {
    // A. stage the block and its halo of 10 (zero outside the image)
    for (int i = tid; i < kDbIn * kDbIn; i += kDbThreads) {
      const int hy = i / kDbIn, hx = i - hy * kDbIn;
      const int qx = x0 + hx - 2 * kDbR, qy = y0 + hy - 2 * kDbR;
      float vx = 0.0f, vy = 0.0f;
      if (qx >= 0 && qx < W && qy >= 0 && qy < H) {
        const size_t o = ((size_t)qy * W + qx) * 3 + ch;
        vx = __ldg(im + o);
        vy = __ldg(ref + o);
      }
      s.x[hy][hx] = (double)vx;
      s.y[hy][hx] = (double)vy;
      const int bx = hx - 2 * kDbR, by = hy - 2 * kDbR;
      if (bx >= 0 && bx < kDbT && by >= 0 && by < kDbT) { s.cx[by][bx] = vx; s.cy[by][bx] = vy; }
    }
    __syncthreads();
    // B. x, x x, x y blurred along x: rows 0..51, columns 0..41 (column c is staged column c + 5); lanes run over
    //    rows (pitch 53 doubles: 16 distinct bank pairs per half-warp)
    for (int i = tid; i < kDbIn * (kDbMid / kRunB); i += kDbThreads) {
      const int grp = i / kDbIn, r = i - grp * kDbIn, c0 = grp * kRunB;
      double xv[kRunB + 2 * kDbR], xx[kRunB + 2 * kDbR], xy[kRunB + 2 * kDbR];
#pragma unroll
      for (int j = 0; j < kRunB + 2 * kDbR; ++j) {
        const double yv = s.y[r][c0 + j];
        xv[j] = s.x[r][c0 + j];
        xx[j] = xv[j] * xv[j];
        xy[j] = xv[j] * yv;
      }
#pragma unroll
      for (int o = 0; o < kRunB; ++o) {
        double a0 = 0, a2 = 0, a4 = 0;
#pragma unroll
        for (int k = 0; k <= 2 * kDbR; ++k) {
          const double g = win.g[k];
          a0 += g * xv[o + k]; a2 += g * xx[o + k]; a4 += g * xy[o + k];
        }
        s.h[0][r][c0 + o] = a0; s.h[1][r][c0 + o] = a2; s.h[2][r][c0 + o] = a4;
      }
    }
    __syncthreads();
    // C. along y, then a, b, c at the 42 x 42 positions (row r is staged row r + 5); lanes run over columns
    for (int i = tid; i < kDbMid * (kDbMid / kRunB); i += kDbThreads) {
      const int grp = i / kDbMid, c = i - grp * kDbMid, r0 = grp * kRunB;
      double mo[3][kRunB];
#pragma unroll
      for (int j3 = 0; j3 < 3; ++j3) {
        double v[kRunB + 2 * kDbR];
#pragma unroll
        for (int j = 0; j < kRunB + 2 * kDbR; ++j) v[j] = s.h[j3][r0 + j][c];
#pragma unroll
        for (int o = 0; o < kRunB; ++o) {
          double acc = 0;
#pragma unroll
          for (int k = 0; k <= 2 * kDbR; ++k) acc += win.g[k] * v[o + k];
          mo[j3][o] = acc;
        }
      }
      const int qx = x0 + c - kDbR;
#pragma unroll
      for (int o = 0; o < kRunB; ++o) {
        const int r = r0 + o, qy = y0 + r - kDbR;
        double va = 0.0, vb = 0.0, vc = 0.0;
        if (qx >= 0 && qx < W && qy >= 0 && qy < H) {
          const size_t oo = ((size_t)qy * W + qx) * 3 + ch;
          const double mx = mo[0][o], my = ref_my[oo], sxx = mo[1][o] - mx * mx, syy = ref_eyy[oo] - my * my,
                       sxy = mo[2][o] - mx * my;
          const double N1 = 2.0 * mx * my + kDbC1, N2 = 2.0 * sxy + kDbC2;
          const double D1 = mx * mx + my * my + kDbC1, D2 = sxx + syy + kDbC2;
          const double r12 = 1.0 / (D1 * D2);
          vb = -N1 * N2 * r12 / D2;
          vc = 2.0 * N1 * r12;
          va = 2.0 * my * N2 * r12 - 2.0 * mx * N1 * N2 * r12 / D1 - 2.0 * mx * vb - my * vc;
        }
        sm[0][r][c] = va; sm[1][r][c] = vb; sm[2][r][c] = vc;
      }
    }
    __syncthreads();
    // D. the maps blurred along x: rows 0..41, block columns 0..31 (block column c is map column c + 5); lanes run
    //    over rows (pitch 43 doubles)
    for (int i = tid; i < kDbMid * (kDbT / kRunD); i += kDbThreads) {
      const int grp = i / kDbMid, r = i - grp * kDbMid, c0 = grp * kRunD;
#pragma unroll
      for (int j3 = 0; j3 < 3; ++j3) {
        double v[kRunD + 2 * kDbR];
#pragma unroll
        for (int j = 0; j < kRunD + 2 * kDbR; ++j) v[j] = sm[j3][r][c0 + j];
#pragma unroll
        for (int o = 0; o < kRunD; ++o) {
          double acc = 0;
#pragma unroll
          for (int k = 0; k <= 2 * kDbR; ++k) acc += win.g[k] * v[o + k];
          gx[j3][r][c0 + o] = acc;
        }
      }
    }
    __syncthreads();
    // E. along y and the pixels' gradient; lanes run over columns
    for (int i = tid; i < kDbT * (kDbT / kRunD); i += kDbThreads) {
      const int grp = i / kDbT, tx = i - grp * kDbT, ty0 = grp * kRunD;
      double bl[3][kRunD];
#pragma unroll
      for (int j3 = 0; j3 < 3; ++j3) {
        double v[kRunD + 2 * kDbR];
#pragma unroll
        for (int j = 0; j < kRunD + 2 * kDbR; ++j) v[j] = gx[j3][ty0 + j][tx];
#pragma unroll
        for (int o = 0; o < kRunD; ++o) {
          double acc = 0;
#pragma unroll
          for (int k = 0; k <= 2 * kDbR; ++k) acc += win.g[k] * v[o + k];
          bl[j3][o] = acc;
        }
      }
      const int px = x0 + tx;
#pragma unroll
      for (int o = 0; o < kRunD; ++o) {
        const int ty = ty0 + o, py = y0 + ty;
        if (px < W && py < H) {
          const double xv = (double)s.cx[ty][tx], yv = (double)s.cy[ty][tx];
          const double dssim = (bl[0][o] + 2.0 * xv * bl[1][o] + yv * bl[2][o]) * inv_n;
          out[(size_t)b * img + ((size_t)py * W + px) * 3 + ch] = (float)(wb * (2.0 * (xv - yv) * inv_n - lambda * dssim));
        }
      }
    }
    __syncthreads();  // the staging buffers are rewritten for the next channel
  }
}

// lambda == 0: the MSE term alone, no window
__global__ void k_mse_backward(const float* __restrict__ imgs, const float* __restrict__ ref, size_t img, int B,
                               const double* __restrict__ weight, float* __restrict__ out) {
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int b = blockIdx.y;
  if (i >= img) return;
  const double wb = weight ? weight[b] : 1.0;
  out[(size_t)b * img + i] = (float)(wb * 2.0 * ((double)imgs[(size_t)b * img + i] - (double)ref[i]) / (double)img);
}

int launch_distortion_backward(const float* imgs, const float* ref, int32_t B, int32_t H, int32_t W,
                               const double* weight, double lambda, float* out, double* ref_planes, cudaStream_t st) {
  if (B == 0) return 0;
  const size_t img = (size_t)H * W * 3;
  if (lambda == 0.0) {
    for (int b0 = 0; b0 < B; b0 += 65535) {
      const int nb = B - b0 < 65535 ? B - b0 : 65535;
      k_mse_backward<<<dim3((unsigned)((img + 255) / 256), nb), 256, 0, st>>>(imgs + (size_t)b0 * img, ref, img, nb,
                                                                             weight ? weight + b0 : nullptr,
                                                                             out + (size_t)b0 * img);
      count_launches(1);
    }
    return 0;
  }
  DbWindow win;
  double g[2 * kDbR + 1], sum = 0.0;
  for (int k = 0; k <= 2 * kDbR; ++k) {  // exp(-(k-5)^2 / (2 * 1.5^2)), normalised
    g[k] = exp(-(double)((k - kDbR) * (k - kDbR)) / (2.0 * 1.5 * 1.5));
    sum += g[k];
  }
  for (int k = 0; k <= 2 * kDbR; ++k) win.g[k] = g[k] / sum;
  if (cudaFuncSetAttribute(k_distortion_backward, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(DbSmem)) !=
      cudaSuccess)
    return -1;
  double* my = ref_planes;
  double* eyy = ref_planes + img;
  const int TX16 = (W + kTile - 1) / kTile, TY16 = (H + kTile - 1) / kTile;
  k_ref_moments<<<TX16 * TY16, kTilePix, 0, st>>>(ref, W, H, TX16, win, my, eyy);
  count_launches(1);
  const int TX = (W + kDbT - 1) / kDbT, TY = (H + kDbT - 1) / kDbT;
  for (int b0 = 0; b0 < B; b0 += 65535) {
    const int nb = B - b0 < 65535 ? B - b0 : 65535;
    k_distortion_backward<<<dim3(TX * TY, nb), kDbThreads, sizeof(DbSmem), st>>>(
        imgs + (size_t)b0 * img, ref, W, H, TX, my, eyy, weight ? weight + b0 : nullptr, lambda, win,
        out + (size_t)b0 * img);
    count_launches(1);
  }
  return 0;
}

}  // namespace gsr
