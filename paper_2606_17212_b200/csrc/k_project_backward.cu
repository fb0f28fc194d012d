// k_project_backward.cu — backward of stages a1-a2 and of the activation (the
// objective reaches the representation through the rendered images; SURVEY.md §8(f)-4 follow-on).
//
// Input: grad_rec [records, 12] = dL/d(rgb[3], rgb with SH residual[3], opacity, A, B, Cq, m_x, m_y) of every
// projected record, summed over the states and pixels that composite it (gsr_render_backward).  Record 2 i + v of
// Gaussian i: v = 0 the geometry without the motion residual (cluster depth 0), v = 1 with it (depth >= 1).
// Output: the gradient with respect to the scene's own parameters,
//     g_gauss   [N, 14]   mean[3], rho[3] (the motion residual vector s_c sum_r b_r q_r), log_scale[3], quat[4] (raw),
//                         opacity_logit
//     g_sh_base [N, K, 3], g_sh_res [N, K, 3]
//     g_cluster [C, 13]   A_c(t) [3,4] row-major (dL/dA0 = it, dL/dA1 = t * it), s_c
// One thread per Gaussian: the forward of DESIGN.md §3.2/§3.3 is recomputed in fp32 for each variant, then walked
// backwards.  The discrete decisions (presence, the culls z > znear and det > 0, the clamp of x/z, y/z at 1.3 lim,
// rgb = max(0, .), tau, radius, rectangle) are constants of the differentiation (reading K1).  The per-cluster sums
// are reduced over the warp when the warp holds one cluster (Gaussians are sorted by cluster) and added with
// float atomics: reproducible up to fp32 summation order.
#include "gsr_internal.h"

namespace gsr {

constexpr float kC1 = 0.4886025119029199f, kK4 = 1.0925484305920792f, kK6 = 0.31539156525252005f,
                kK8 = 0.5462742152960396f, kK9 = 0.5900435899266435f, kK10 = 2.890611442640554f,
                kK11 = 0.4570457994644658f, kK12 = 0.3731763325901154f, kK14 = 1.445305721320277f;

template <int K>
__device__ __forceinline__ void sh_values(float x, float y, float z, float* Y) {
  Y[0] = 0.28209479177387814f;
  if (K > 1) { Y[1] = kC1 * y; Y[2] = kC1 * z; Y[3] = kC1 * x; }
  if (K > 4) {
    Y[4] = kK4 * x * y; Y[5] = kK4 * y * z; Y[6] = kK6 * (3.0f * z * z - 1.0f); Y[7] = kK4 * x * z;
    Y[8] = kK8 * (x * x - y * y);
  }
  if (K > 9) {
    Y[9] = kK9 * y * (3.0f * x * x - y * y); Y[10] = kK10 * x * y * z; Y[11] = kK11 * y * (5.0f * z * z - 1.0f);
    Y[12] = kK12 * (5.0f * z * z * z - 3.0f * z); Y[13] = kK11 * x * (5.0f * z * z - 1.0f);
    Y[14] = kK14 * (x * x - y * y) * z; Y[15] = kK9 * x * (x * x - 3.0f * y * y);
  }
}

// sum_j dY[j] * grad Y_j(x, y, z), x, y, z taken as independent variables
template <int K>
__device__ __forceinline__ void sh_grad_dot(float x, float y, float z, const float* dY, float* g) {
  g[0] = g[1] = g[2] = 0.0f;
  if (K > 1) { g[1] += kC1 * dY[1]; g[2] += kC1 * dY[2]; g[0] += kC1 * dY[3]; }
  if (K > 4) {
    g[0] += kK4 * (y * dY[4] + z * dY[7]) + 2.0f * kK8 * x * dY[8];
    g[1] += kK4 * (x * dY[4] + z * dY[5]) - 2.0f * kK8 * y * dY[8];
    g[2] += kK4 * (y * dY[5] + x * dY[7]) + 6.0f * kK6 * z * dY[6];
  }
  if (K > 9) {
    const float xx = x * x, yy = y * y, zz = z * z, f5 = 5.0f * zz - 1.0f;
    g[0] += 6.0f * kK9 * x * y * dY[9] + kK10 * y * z * dY[10] + kK11 * f5 * dY[13] + 2.0f * kK14 * x * z * dY[14] +
            3.0f * kK9 * (xx - yy) * dY[15];
    g[1] += 3.0f * kK9 * (xx - yy) * dY[9] + kK10 * x * z * dY[10] + kK11 * f5 * dY[11] - 2.0f * kK14 * y * z * dY[14] -
            6.0f * kK9 * x * y * dY[15];
    g[2] += kK10 * x * y * dY[10] + 10.0f * kK11 * z * (y * dY[11] + x * dY[13]) + kK12 * (15.0f * zz - 3.0f) * dY[12] +
            kK14 * (xx - yy) * dY[14];
  }
}

struct PbArgs {
  const float* grad_rec;  // [2N, 12]
  float* g_gauss;         // [N, 14]
  float* g_shb;           // [N, K, 3]
  float* g_shr;           // [N, K, 3]
  float* g_cluster;       // [C, 13]
};

// One variant: geometry mean `mu`; gc0 / gc1 = dL/d(first / second colour) (gc1 only for the variant with the
// residual), gq = dL/d(opacity, A, B, Cq, m_x, m_y).  Adds to dmu, dS6 (dL/dSigma, the 9 entries folded onto the 6
// stored ones), dopac and the SH gradients of Gaussian i (its rows of the CTA's shared tile).  Returns false if the
// variant is culled.
template <int K>
__device__ __forceinline__ bool variant_backward(const DeviceScene& sc, const FrameParams& fp, int i, const float* mu,
                                                 const float* S6, bool with_res, const float* gc0, const float* gc1,
                                                 const float* gq, float* dmu, float* dS6, float& dopac,
                                                 float* shb_row, float* shr_row, int n_dsh = 0,
                                                 float* const* dsh_rows = nullptr) {
  const float* Rw = fp.R;
  float pc[3];
#pragma unroll
  for (int k = 0; k < 3; ++k) pc[k] = Rw[3 * k] * mu[0] + Rw[3 * k + 1] * mu[1] + Rw[3 * k + 2] * mu[2] + fp.t[k];
  const float z = pc[2];
  if (!(z > fp.znear)) return false;
  const float rz = 1.0f / z, txz = pc[0] * rz, tyz = pc[1] * rz;
  const float limx = ((0.5f * (float)fp.W) / fp.fx) * 1.3f, limy = ((0.5f * (float)fp.H) / fp.fy) * 1.3f;
  const bool in_x = txz >= -limx && txz <= limx, in_y = tyz >= -limy && tyz <= limy;
  const float cxz = fminf(limx, fmaxf(-limx, txz)), cyz = fminf(limy, fmaxf(-limy, tyz));
  const float xt = cxz * z, yt = cyz * z;
  const float J00 = fp.fx * rz, J02 = -fp.fx * xt * rz * rz, J11 = fp.fy * rz, J12 = -fp.fy * yt * rz * rz;
  float M0[3], M1[3], v0[3], v1[3];
#pragma unroll
  for (int k = 0; k < 3; ++k) {
    M0[k] = J00 * Rw[k] + J02 * Rw[6 + k];
    M1[k] = J11 * Rw[3 + k] + J12 * Rw[6 + k];
  }
  const float S[9] = {S6[0], S6[1], S6[2], S6[1], S6[3], S6[4], S6[2], S6[4], S6[5]};
#pragma unroll
  for (int r = 0; r < 3; ++r) {
    v0[r] = S[3 * r] * M0[0] + S[3 * r + 1] * M0[1] + S[3 * r + 2] * M0[2];
    v1[r] = S[3 * r] * M1[0] + S[3 * r + 1] * M1[1] + S[3 * r + 2] * M1[2];
  }
  const float ca = M0[0] * v0[0] + M0[1] * v0[1] + M0[2] * v0[2] + 0.3f;
  const float cb = M0[0] * v1[0] + M0[1] * v1[1] + M0[2] * v1[2];
  const float cc = M1[0] * v1[0] + M1[1] * v1[1] + M1[2] * v1[2] + 0.3f;
  const float det = ca * cc - cb * cb;
  if (!(det > 0.0f)) return false;

  // ---- colour: rgb = max(0, 0.5 + sum_j Y_j coef_j)
  float dmu_c[3] = {0.f, 0.f, 0.f};
  {
    const float dvx = mu[0] - fp.cam_centre[0], dvy = mu[1] - fp.cam_centre[1], dvz = mu[2] - fp.cam_centre[2];
    const float inv = rsqrtf(dvx * dvx + dvy * dvy + dvz * dvz);
    const float dx = dvx * inv, dy = dvy * inv, dz = dvz * inv;
    float Y[K];
    sh_values<K>(dx, dy, dz, Y);
    float s0[3] = {0.5f, 0.5f, 0.5f}, s1[3] = {0.f, 0.f, 0.f};
    constexpr int n4 = (3 * K + 3) / 4;
#pragma unroll
    for (int w4 = 0; w4 < n4; ++w4) {
      const float4 b4 = __ldg(sc.sh_base + (size_t)w4 * sc.N + i);
      float vb[4] = {b4.x, b4.y, b4.z, b4.w};
      for (int l = 0; l < n_dsh; ++l) {  // colour refinements of the delivered levels 1..n_dsh (reading I3)
        const float4 dl = __ldg(sc.d_sh + ((size_t)l * n4 + w4) * sc.N + i);
        vb[0] += dl.x; vb[1] += dl.y; vb[2] += dl.z; vb[3] += dl.w;
      }
      float vr[4] = {0.f, 0.f, 0.f, 0.f};
      if (with_res) {
        const float4 r4 = __ldg(sc.sh_res + (size_t)w4 * sc.N + i);
        vr[0] = r4.x; vr[1] = r4.y; vr[2] = r4.z; vr[3] = r4.w;
      }
#pragma unroll
      for (int e = 0; e < 4; ++e) {
        const int flat = w4 * 4 + e;
        if (flat < 3 * K) {
          s0[flat % 3] = fmaf(Y[flat / 3], vb[e], s0[flat % 3]);
          s1[flat % 3] = fmaf(Y[flat / 3], vr[e], s1[flat % 3]);
        }
      }
    }
    float d0[3], d1[3];
    bool any = false;
#pragma unroll
    for (int ch = 0; ch < 3; ++ch) {
      d0[ch] = s0[ch] > 0.0f ? gc0[ch] : 0.0f;
      d1[ch] = (with_res && s0[ch] + s1[ch] > 0.0f) ? gc1[ch] : 0.0f;
      any |= d0[ch] != 0.0f || d1[ch] != 0.0f;
    }
    if (any) {
      float dY[K];
#pragma unroll
      for (int j = 0; j < K; ++j) dY[j] = 0.0f;
#pragma unroll
      for (int w4 = 0; w4 < n4; ++w4) {
        const float4 b4 = __ldg(sc.sh_base + (size_t)w4 * sc.N + i);
        float vb[4] = {b4.x, b4.y, b4.z, b4.w};
        for (int l = 0; l < n_dsh; ++l) {
          const float4 dl = __ldg(sc.d_sh + ((size_t)l * n4 + w4) * sc.N + i);
          vb[0] += dl.x; vb[1] += dl.y; vb[2] += dl.z; vb[3] += dl.w;
        }
        float vr[4] = {0.f, 0.f, 0.f, 0.f};
        if (with_res) {
          const float4 r4 = __ldg(sc.sh_res + (size_t)w4 * sc.N + i);
          vr[0] = r4.x; vr[1] = r4.y; vr[2] = r4.z; vr[3] = r4.w;
        }
#pragma unroll
        for (int e = 0; e < 4; ++e) {
          const int flat = w4 * 4 + e;
          if (flat < 3 * K) {
            const int j = flat / 3, ch = flat % 3;
            dY[j] += d0[ch] * vb[e] + d1[ch] * (vb[e] + vr[e]);
            shb_row[flat] += Y[j] * (d0[ch] + d1[ch]);
            if (with_res) shr_row[flat] += Y[j] * d1[ch];
            for (int l = 0; l < n_dsh; ++l) dsh_rows[l][flat] += Y[j] * (d0[ch] + d1[ch]);
          }
        }
      }
      float gd[3];
      sh_grad_dot<K>(dx, dy, dz, dY, gd);
      const float dot = dx * gd[0] + dy * gd[1] + dz * gd[2];
      dmu_c[0] = (gd[0] - dx * dot) * inv;
      dmu_c[1] = (gd[1] - dy * dot) * inv;
      dmu_c[2] = (gd[2] - dz * dot) * inv;
    }
  }
  dopac += gq[0];

  // ---- conic = X^-1, X = [[a, b], [b, c]]: dL/dX = -Q Gs Q with Gs the symmetric gradient with respect to Q
  const float rdet = 1.0f / det;
  const float q00 = cc * rdet, q01 = -cb * rdet, q11 = ca * rdet;
  const float g00 = 0.5f * gq[1], h = 0.5f * gq[2], g11 = 0.5f * gq[3];
  const float t00 = q00 * g00 + q01 * h, t01 = q00 * h + q01 * g11, t10 = q01 * g00 + q11 * h, t11 = q01 * h + q11 * g11;
  const float da = -(t00 * q00 + t01 * q01), db = -2.0f * (t00 * q01 + t01 * q11), dc = -(t10 * q01 + t11 * q11);
  // Sigma' = M Sigma M^T: dL/dSigma (9 entries folded onto the 6 stored), dL/dM
  dS6[0] += da * M0[0] * M0[0] + db * M0[0] * M1[0] + dc * M1[0] * M1[0];
  dS6[3] += da * M0[1] * M0[1] + db * M0[1] * M1[1] + dc * M1[1] * M1[1];
  dS6[5] += da * M0[2] * M0[2] + db * M0[2] * M1[2] + dc * M1[2] * M1[2];
  dS6[1] += 2.0f * (da * M0[0] * M0[1] + dc * M1[0] * M1[1]) + db * (M0[0] * M1[1] + M0[1] * M1[0]);
  dS6[2] += 2.0f * (da * M0[0] * M0[2] + dc * M1[0] * M1[2]) + db * (M0[0] * M1[2] + M0[2] * M1[0]);
  dS6[4] += 2.0f * (da * M0[1] * M0[2] + dc * M1[1] * M1[2]) + db * (M0[1] * M1[2] + M0[2] * M1[1]);
  float dJ00 = 0.f, dJ02 = 0.f, dJ11 = 0.f, dJ12 = 0.f;
#pragma unroll
  for (int k = 0; k < 3; ++k) {
    const float dM0 = 2.0f * da * v0[k] + db * v1[k], dM1 = 2.0f * dc * v1[k] + db * v0[k];
    dJ00 += dM0 * Rw[k]; dJ02 += dM0 * Rw[6 + k];
    dJ11 += dM1 * Rw[3 + k]; dJ12 += dM1 * Rw[6 + k];
  }
  float drz = fp.fx * dJ00 + fp.fy * dJ11 - 2.0f * rz * (fp.fx * xt * dJ02 + fp.fy * yt * dJ12);
  const float dxt = -fp.fx * rz * rz * dJ02, dyt = -fp.fy * rz * rz * dJ12;
  float dz = cxz * dxt + cyz * dyt;
  float dtxz = fp.fx * gq[4], dtyz = fp.fy * gq[5];
  if (in_x) dtxz += z * dxt;
  if (in_y) dtyz += z * dyt;
  const float dpc0 = rz * dtxz, dpc1 = rz * dtyz;
  drz += pc[0] * dtxz + pc[1] * dtyz;
  dz -= rz * rz * drz;
#pragma unroll
  for (int k = 0; k < 3; ++k) dmu[k] += Rw[k] * dpc0 + Rw[3 + k] * dpc1 + Rw[6 + k] * dz + dmu_c[k];
  return true;
}

constexpr int kPbThreads = 64;

template <int K>
__global__ void __launch_bounds__(kPbThreads) k_project_backward(DeviceScene sc, FrameParams fp, PbArgs a) {
  // the SH gradients of the CTA's Gaussians: [thread][3K (+1: conflict-free rows)], written out coalesced at the end
  constexpr int kRow = 3 * K + 1;
  __shared__ float s_shb[kPbThreads * kRow], s_shr[kPbThreads * kRow];
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int lane = threadIdx.x & 31;
  const bool live = i < sc.N;
  float* const shb_row = s_shb + threadIdx.x * kRow;
  float* const shr_row = s_shr + threadIdx.x * kRow;
#pragma unroll
  for (int f = 0; f < 3 * K; ++f) { shb_row[f] = 0.0f; shr_row[f] = 0.0f; }
  int c = -1;
  float cl13[13];
#pragma unroll
  for (int k = 0; k < 13; ++k) cl13[k] = 0.0f;
  if (live) {
    const float4 g0 = __ldg(sc.g0 + i), g1 = __ldg(sc.g1 + i), g2 = __ldg(sc.g2 + i);
    const uint32_t bits = __float_as_uint(g2.w);
    c = (int)(bits >> 2);
    const int lvl = (int)(bits & 3u);
    const float S6[6] = {g1.x, g1.y, g1.z, g2.x, g2.y, g2.z};
    // ---- Eq. (1)
    float A[12];
#pragma unroll
    for (int k = 0; k < 12; ++k) A[k] = fmaf(fp.time, __ldg(sc.A1 + 12 * c + k), __ldg(sc.A0 + 12 * c + k));
    float p[3], acc[3] = {0.f, 0.f, 0.f}, muB[3];
#pragma unroll
    for (int k = 0; k < 3; ++k) p[k] = A[4 * k] * g0.x + A[4 * k + 1] * g0.y + A[4 * k + 2] * g0.z + A[4 * k + 3];
    {
      uint32_t w = 0;
      for (int r = 0; r < sc.R; ++r) {
#pragma unroll
        for (int k = 0; k < 3; ++k) {
          const int byte = r * 3 + k;
          if ((byte & 3) == 0) w = __ldg(sc.qw + (size_t)(byte >> 2) * sc.N + i);
          acc[k] = fmaf(fp.basis[r], (float)(int)(int8_t)((w >> ((byte & 3) * 8)) & 0xFFu), acc[k]);
        }
      }
    }
    const float s_c = __ldg(sc.mscale + c);
#pragma unroll
    for (int k = 0; k < 3; ++k) muB[k] = fmaf(s_c, acc[k], p[k]);

    float dp[3] = {0.f, 0.f, 0.f}, drho[3] = {0.f, 0.f, 0.f}, dS6[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f}, dopac = 0.0f;
    const float zero3[3] = {0.f, 0.f, 0.f};
    if (lvl == 0) {  // variant A: record 2 i, one colour (the first triple)
      float g[12];
      const float4* gp = reinterpret_cast<const float4*>(a.grad_rec + 12 * (size_t)(2 * i));
#pragma unroll
      for (int q = 0; q < 3; ++q) { const float4 v = __ldg(gp + q); g[4 * q] = v.x; g[4 * q + 1] = v.y; g[4 * q + 2] = v.z; g[4 * q + 3] = v.w; }
      variant_backward<K>(sc, fp, i, p, S6, false, g, zero3, g + 6, dp, dS6, dopac, shb_row, shr_row);
    }
    {  // variant B: record 2 i + 1, colours without / with the SH residual
      float g[12];
      const float4* gp = reinterpret_cast<const float4*>(a.grad_rec + 12 * (size_t)(2 * i + 1));
#pragma unroll
      for (int q = 0; q < 3; ++q) { const float4 v = __ldg(gp + q); g[4 * q] = v.x; g[4 * q + 1] = v.y; g[4 * q + 2] = v.z; g[4 * q + 3] = v.w; }
      variant_backward<K>(sc, fp, i, muB, S6, true, g, g + 3, g + 6, drho, dS6, dopac, shb_row, shr_row);
    }
    // ---- deformation: mu_A = p, mu_B = p + rho
#pragma unroll
    for (int k = 0; k < 3; ++k) dp[k] += drho[k];
    float* out = a.g_gauss + 14 * (size_t)i;
#pragma unroll
    for (int j = 0; j < 3; ++j) out[j] = A[j] * dp[0] + A[4 + j] * dp[1] + A[8 + j] * dp[2];
#pragma unroll
    for (int k = 0; k < 3; ++k) out[3 + k] = drho[k];
#pragma unroll
    for (int k = 0; k < 3; ++k) {
      cl13[4 * k] = dp[k] * g0.x; cl13[4 * k + 1] = dp[k] * g0.y; cl13[4 * k + 2] = dp[k] * g0.z; cl13[4 * k + 3] = dp[k];
    }
    cl13[12] = drho[0] * acc[0] + drho[1] * acc[1] + drho[2] * acc[2];
    // ---- activation: Sigma = Mm Mm^T, Mm = Rm diag(exp(ls)); opacity = sigmoid(logit)
    const float4 rq = __ldg(sc.raw_quat + i), rl = __ldg(sc.raw_ls + i);
    const float qn = sqrtf(rq.x * rq.x + rq.y * rq.y + rq.z * rq.z + rq.w * rq.w), rqn = 1.0f / qn;
    const float w = rq.x * rqn, x = rq.y * rqn, y = rq.z * rqn, z = rq.w * rqn;
    const float Rm[9] = {1.f - 2.f * (y * y + z * z), 2.f * (x * y - w * z), 2.f * (x * z + w * y),
                         2.f * (x * y + w * z), 1.f - 2.f * (x * x + z * z), 2.f * (y * z - w * x),
                         2.f * (x * z - w * y), 2.f * (y * z + w * x), 1.f - 2.f * (x * x + y * y)};
    const float s3[3] = {expf(rl.x), expf(rl.y), expf(rl.z)};
    // dL/dMm = (G + G^T) Mm with the folded dS6: (G + G^T) has 2 dS6 on the diagonal entries, dS6 off the diagonal
    const float Gs[9] = {2.f * dS6[0], dS6[1], dS6[2], dS6[1], 2.f * dS6[3], dS6[4], dS6[2], dS6[4], 2.f * dS6[5]};
    float dRm[9];
#pragma unroll
    for (int k = 0; k < 3; ++k) {
      float ds = 0.0f;
#pragma unroll
      for (int r = 0; r < 3; ++r) {
        const float dMm = (Gs[3 * r] * Rm[k] + Gs[3 * r + 1] * Rm[3 + k] + Gs[3 * r + 2] * Rm[6 + k]) * s3[k];
        ds += dMm * Rm[3 * r + k];
        dRm[3 * r + k] = dMm * s3[k];
      }
      out[6 + k] = ds * s3[k];
    }
    const float dw = 2.f * (-z * dRm[1] + y * dRm[2] + z * dRm[3] - x * dRm[5] - y * dRm[6] + x * dRm[7]);
    const float dx = 2.f * (y * dRm[1] + z * dRm[2] + y * dRm[3] - 2.f * x * dRm[4] - w * dRm[5] + z * dRm[6] + w * dRm[7] - 2.f * x * dRm[8]);
    const float dy = 2.f * (-2.f * y * dRm[0] + x * dRm[1] + w * dRm[2] + x * dRm[3] + z * dRm[5] - w * dRm[6] + z * dRm[7] - 2.f * y * dRm[8]);
    const float dz = 2.f * (-2.f * z * dRm[0] - w * dRm[1] + x * dRm[2] + w * dRm[3] - 2.f * z * dRm[4] + y * dRm[5] + x * dRm[6] + y * dRm[7]);
    const float qd = w * dw + x * dx + y * dy + z * dz;
    out[9] = (dw - w * qd) * rqn;
    out[10] = (dx - x * qd) * rqn;
    out[11] = (dy - y * qd) * rqn;
    out[12] = (dz - z * qd) * rqn;
    out[13] = dopac * g0.w * (1.0f - g0.w);
  }
  // ---- the CTA's SH gradients: rows i0 .. i0 + 63 are contiguous in g_sh_base / g_sh_res
  __syncthreads();
  {
    const size_t i0 = (size_t)blockIdx.x * kPbThreads;
    const int rows = sc.N - (int)i0 < kPbThreads ? sc.N - (int)i0 : kPbThreads;
    for (int f = threadIdx.x; f < rows * 3 * K; f += kPbThreads) {
      const int r = f / (3 * K), col = f - r * (3 * K);
      a.g_shb[i0 * 3 * K + f] = s_shb[r * kRow + col];
      a.g_shr[i0 * 3 * K + f] = s_shr[r * kRow + col];
    }
  }
  // ---- per-cluster sums: over the warp when it holds one cluster, else lane by lane
  const int c0 = __shfl_sync(0xffffffffu, c, 0);
  if (__all_sync(0xffffffffu, c == c0)) {
    if (c0 < 0) return;
#pragma unroll
    for (int k = 0; k < 13; ++k) {
      float v = cl13[k];
#pragma unroll
      for (int off = 16; off > 0; off >>= 1) v += __shfl_xor_sync(0xffffffffu, v, off);
      if (lane == 0 && v != 0.0f) atomicAdd(a.g_cluster + 13 * (size_t)c0 + k, v);
    }
  } else if (live) {
#pragma unroll
    for (int k = 0; k < 13; ++k)
      if (cl13[k] != 0.0f) atomicAdd(a.g_cluster + 13 * (size_t)c + k, cl13[k]);
  }
}

// ------------------------------------------------------------------------------------------------
// The full representation: four records per Gaussian, one per delivered depth v = 0..3
// (record 4 i + v, one colour each), with position residual levels, per-level attribute and colour refinements and,
// optionally, the affine on the covariance.

// Backward of the activation for one set of raw attributes: dS6 = dL/dSigma folded onto the 6
// stored entries, dopac = dL/d(opacity), opac = the activated opacity -> out8 = d/d(log_scale[3], quat[4], logit)
__device__ __forceinline__ void activation_backward(const float4 rq, const float4 rl, const float* dS6, float dopac,
                                                    float opac, float* out8) {
  const float qn = sqrtf(rq.x * rq.x + rq.y * rq.y + rq.z * rq.z + rq.w * rq.w), rqn = 1.0f / qn;
  const float w = rq.x * rqn, x = rq.y * rqn, y = rq.z * rqn, z = rq.w * rqn;
  const float Rm[9] = {1.f - 2.f * (y * y + z * z), 2.f * (x * y - w * z), 2.f * (x * z + w * y),
                       2.f * (x * y + w * z), 1.f - 2.f * (x * x + z * z), 2.f * (y * z - w * x),
                       2.f * (x * z - w * y), 2.f * (y * z + w * x), 1.f - 2.f * (x * x + y * y)};
  const float s3[3] = {expf(rl.x), expf(rl.y), expf(rl.z)};
  const float Gs[9] = {2.f * dS6[0], dS6[1], dS6[2], dS6[1], 2.f * dS6[3], dS6[4], dS6[2], dS6[4], 2.f * dS6[5]};
  float dRm[9];
#pragma unroll
  for (int k = 0; k < 3; ++k) {
    float ds = 0.0f;
#pragma unroll
    for (int r = 0; r < 3; ++r) {
      const float dMm = (Gs[3 * r] * Rm[k] + Gs[3 * r + 1] * Rm[3 + k] + Gs[3 * r + 2] * Rm[6 + k]) * s3[k];
      ds += dMm * Rm[3 * r + k];
      dRm[3 * r + k] = dMm * s3[k];
    }
    out8[k] = ds * s3[k];
  }
  const float dw = 2.f * (-z * dRm[1] + y * dRm[2] + z * dRm[3] - x * dRm[5] - y * dRm[6] + x * dRm[7]);
  const float dx = 2.f * (y * dRm[1] + z * dRm[2] + y * dRm[3] - 2.f * x * dRm[4] - w * dRm[5] + z * dRm[6] + w * dRm[7] - 2.f * x * dRm[8]);
  const float dy = 2.f * (-2.f * y * dRm[0] + x * dRm[1] + w * dRm[2] + x * dRm[3] + z * dRm[5] - w * dRm[6] + z * dRm[7] - 2.f * y * dRm[8]);
  const float dz = 2.f * (-2.f * z * dRm[0] - w * dRm[1] + x * dRm[2] + w * dRm[3] - 2.f * z * dRm[4] + y * dRm[5] + x * dRm[6] + y * dRm[7]);
  const float qd = w * dw + x * dx + y * dy + z * dz;
  out8[3] = (dw - w * qd) * rqn;
  out8[4] = (dx - x * qd) * rqn;
  out8[5] = (dy - y * qd) * rqn;
  out8[6] = (dz - z * qd) * rqn;
  out8[7] = dopac * opac * (1.0f - opac);
}

// Reading I4: Su = L Sg L^T, L = the 3x3 part of A (row-major 3x4).  Forward.
__device__ __forceinline__ void affine_cov_forward(const float* A, const float* S6, float* Su6) {
  const float Sf[9] = {S6[0], S6[1], S6[2], S6[1], S6[3], S6[4], S6[2], S6[4], S6[5]};
  float LS[9];
#pragma unroll
  for (int a = 0; a < 3; ++a)
#pragma unroll
    for (int b = 0; b < 3; ++b) LS[3 * a + b] = A[4 * a] * Sf[b] + A[4 * a + 1] * Sf[3 + b] + A[4 * a + 2] * Sf[6 + b];
  int o = 0;
#pragma unroll
  for (int a = 0; a < 3; ++a)
#pragma unroll
    for (int b = a; b < 3; ++b) Su6[o++] = LS[3 * a] * A[4 * b] + LS[3 * a + 1] * A[4 * b + 1] + LS[3 * a + 2] * A[4 * b + 2];
}

// ... and backward: dSu6 (folded) -> dSg6 (folded) = L^T G L, and dL/dL = (G + G^T) L Sg added to dA (3x4 row-major)
__device__ __forceinline__ void affine_cov_backward(const float* A, const float* S6, const float* dSu6, float* dSg6,
                                                    float* dA) {
  const float Sf[9] = {S6[0], S6[1], S6[2], S6[1], S6[3], S6[4], S6[2], S6[4], S6[5]};
  // the symmetric part of G: diagonal entries as they are, off-diagonal ones halved
  const float G[9] = {dSu6[0], 0.5f * dSu6[1], 0.5f * dSu6[2], 0.5f * dSu6[1], dSu6[3], 0.5f * dSu6[4],
                      0.5f * dSu6[2], 0.5f * dSu6[4], dSu6[5]};
  float LS[9], GL[9];
#pragma unroll
  for (int a = 0; a < 3; ++a)
#pragma unroll
    for (int b = 0; b < 3; ++b) {
      LS[3 * a + b] = A[4 * a] * Sf[b] + A[4 * a + 1] * Sf[3 + b] + A[4 * a + 2] * Sf[6 + b];
      GL[3 * a + b] = G[3 * a] * A[b] + G[3 * a + 1] * A[4 + b] + G[3 * a + 2] * A[8 + b];  // (G L)_ab
    }
#pragma unroll
  for (int r = 0; r < 3; ++r)
#pragma unroll
    for (int c = 0; c < 3; ++c) dA[4 * r + c] += 2.0f * (G[3 * r] * LS[c] + G[3 * r + 1] * LS[3 + c] + G[3 * r + 2] * LS[6 + c]);
  float T[9];  // L^T (G L)
#pragma unroll
  for (int a = 0; a < 3; ++a)
#pragma unroll
    for (int b = 0; b < 3; ++b) T[3 * a + b] = A[a] * GL[b] + A[4 + a] * GL[3 + b] + A[8 + a] * GL[6 + b];
  dSg6[0] = T[0]; dSg6[1] = 2.0f * T[1]; dSg6[2] = 2.0f * T[2]; dSg6[3] = T[4]; dSg6[4] = 2.0f * T[5]; dSg6[5] = T[8];
}

struct Pb4Args {
  const float* grad_rec;  // [4N, 12]
  float* g_gauss;         // [N, 14]
  float* g_shb;           // [N, K, 3]
  float* g_shr;           // [N, K, 3]
  float* g_cluster;       // [C, 13]
  float* g_delta;         // [N, 6] delta2.xyz, delta3.xyz, or nullptr
  float* g_attr;          // [3][N, 8] per refinement level: log_scale[3], quat[4], logit, or nullptr
  float* g_dsh;           // [3][N, K, 3], or nullptr
};

constexpr int kPb4Threads = 32;

template <int K>
__global__ void __launch_bounds__(kPb4Threads) k_project_backward4(DeviceScene sc, FrameParams fp, Pb4Args a) {
  constexpr int kRow = 3 * K + 1;
  constexpr int n4 = (3 * K + 3) / 4;
  // rows of the CTA's Gaussians: sh_base, sh_res, and the three colour refinement levels
  __shared__ float s_rows[5][kPb4Threads * kRow];
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int lane = threadIdx.x & 31;
  const bool live = i < sc.N;
  float* const shb_row = s_rows[0] + threadIdx.x * kRow;
  float* const shr_row = s_rows[1] + threadIdx.x * kRow;
  float* const dsh_rows[3] = {s_rows[2] + threadIdx.x * kRow, s_rows[3] + threadIdx.x * kRow, s_rows[4] + threadIdx.x * kRow};
#pragma unroll
  for (int r = 0; r < 5; ++r)
    for (int f = 0; f < 3 * K; ++f) s_rows[r][threadIdx.x * kRow + f] = 0.0f;
  int c = -1;
  float cl13[13];
#pragma unroll
  for (int k = 0; k < 13; ++k) cl13[k] = 0.0f;
  if (live) {
    const float4 g0 = __ldg(sc.g0 + i), g1 = __ldg(sc.g1 + i), g2 = __ldg(sc.g2 + i);
    const uint32_t bits = __float_as_uint(g2.w);
    c = (int)(bits >> 2);
    const int lvl = (int)(bits & 3u);
    // ---- Eq. (1) with the position residual levels: mu_0 = p, mu_1 = p + rho, mu_2 = mu_1 + delta2, mu_3 = mu_2 + delta3
    float A[12];
#pragma unroll
    for (int k = 0; k < 12; ++k) A[k] = fmaf(fp.time, __ldg(sc.A1 + 12 * c + k), __ldg(sc.A0 + 12 * c + k));
    float mu[4][3], acc[3] = {0.f, 0.f, 0.f};
#pragma unroll
    for (int k = 0; k < 3; ++k) mu[0][k] = A[4 * k] * g0.x + A[4 * k + 1] * g0.y + A[4 * k + 2] * g0.z + A[4 * k + 3];
    {
      uint32_t w = 0;
      for (int r = 0; r < sc.R; ++r) {
#pragma unroll
        for (int k = 0; k < 3; ++k) {
          const int byte = r * 3 + k;
          if ((byte & 3) == 0) w = __ldg(sc.qw + (size_t)(byte >> 2) * sc.N + i);
          acc[k] = fmaf(fp.basis[r], (float)(int)(int8_t)((w >> ((byte & 3) * 8)) & 0xFFu), acc[k]);
        }
      }
    }
    const float s_c = __ldg(sc.mscale + c);
#pragma unroll
    for (int k = 0; k < 3; ++k) {
      mu[1][k] = fmaf(s_c, acc[k], mu[0][k]);
      mu[2][k] = mu[1][k] + __ldg(sc.delta + (size_t)k * sc.N + i);
      mu[3][k] = mu[2][k] + __ldg(sc.delta + (size_t)(3 + k) * sc.N + i);
    }
    const bool attr = sc.g1v != nullptr;
    float dmu_all[3] = {0.f, 0.f, 0.f}, drho[3] = {0.f, 0.f, 0.f}, dd2[3] = {0.f, 0.f, 0.f}, dd3[3] = {0.f, 0.f, 0.f};
    float dA[12];
#pragma unroll
    for (int k = 0; k < 12; ++k) dA[k] = 0.0f;
    float base8[8], lev[3][8], dS6sum[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f}, dopac_sum = 0.0f;
#pragma unroll
    for (int k = 0; k < 8; ++k) { base8[k] = 0.0f; lev[0][k] = 0.0f; lev[1][k] = 0.0f; lev[2][k] = 0.0f; }
    const float zero3[3] = {0.f, 0.f, 0.f};
#pragma unroll
    for (int v = 0; v < 4; ++v) {
      if (v < lvl) continue;  // a level-l Gaussian has the variants v >= l only
      float S6[6] = {g1.x, g1.y, g1.z, g2.x, g2.y, g2.z}, opac = g0.w;
      if (attr) {  // the attributes of delivered depth v (reading I2)
        const float4 h1 = __ldg(sc.g1v + (size_t)v * sc.N + i), h2 = __ldg(sc.g2v + (size_t)v * sc.N + i);
        S6[0] = h1.x; S6[1] = h1.y; S6[2] = h1.z; S6[3] = h2.x; S6[4] = h2.y; S6[5] = h2.z;
        opac = __ldg(sc.opv + (size_t)v * sc.N + i);
      }
      float Su[6];
      if (sc.affine_cov) affine_cov_forward(A, S6, Su);
      else {
#pragma unroll
        for (int k = 0; k < 6; ++k) Su[k] = S6[k];
      }
      float g[12];
      const float4* gp = reinterpret_cast<const float4*>(a.grad_rec + 12 * (size_t)(4 * i + v));
#pragma unroll
      for (int q = 0; q < 3; ++q) { const float4 t4 = __ldg(gp + q); g[4 * q] = t4.x; g[4 * q + 1] = t4.y; g[4 * q + 2] = t4.z; g[4 * q + 3] = t4.w; }
      float dmu[3] = {0.f, 0.f, 0.f}, dSu[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f}, dop = 0.0f;
      // one colour per record (columns 0..2): at depth 3 it includes the SH residual
      const bool ok = variant_backward<K>(sc, fp, i, mu[v], Su, v == 3, v == 3 ? zero3 : g, v == 3 ? g : zero3, g + 6, dmu,
                                          dSu, dop, shb_row, shr_row, sc.d_sh ? v : 0, dsh_rows);
      if (!ok) continue;
      float dSg[6];
      if (sc.affine_cov) affine_cov_backward(A, S6, dSu, dSg, dA);
      else {
#pragma unroll
        for (int k = 0; k < 6; ++k) dSg[k] = dSu[k];
      }
#pragma unroll
      for (int k = 0; k < 3; ++k) {
        dmu_all[k] += dmu[k];
        if (v >= 1) drho[k] += dmu[k];
        if (v >= 2) dd2[k] += dmu[k];
        if (v >= 3) dd3[k] += dmu[k];
      }
      if (attr) {
        float gv[8];
        activation_backward(__ldg(sc.raw_quat_v + (size_t)v * sc.N + i), __ldg(sc.raw_ls_v + (size_t)v * sc.N + i), dSg, dop,
                            opac, gv);
#pragma unroll
        for (int k = 0; k < 8; ++k) {
          base8[k] += gv[k];
#pragma unroll
          for (int l = 0; l < 3; ++l)
            if (l < v) lev[l][k] += gv[k];  // the residual of level l + 1 is part of every depth >= l + 1
        }
      } else {
#pragma unroll
        for (int k = 0; k < 6; ++k) dS6sum[k] += dSg[k];
        dopac_sum += dop;
      }
    }
    if (!attr) activation_backward(__ldg(sc.raw_quat + i), __ldg(sc.raw_ls + i), dS6sum, dopac_sum, g0.w, base8);
    float* out = a.g_gauss + 14 * (size_t)i;
#pragma unroll
    for (int j = 0; j < 3; ++j) out[j] = A[j] * dmu_all[0] + A[4 + j] * dmu_all[1] + A[8 + j] * dmu_all[2];
#pragma unroll
    for (int k = 0; k < 3; ++k) out[3 + k] = drho[k];
#pragma unroll
    for (int k = 0; k < 8; ++k) out[6 + k] = base8[k];
    if (a.g_delta) {
#pragma unroll
      for (int k = 0; k < 3; ++k) {  // zero where the scene has no such residual
        a.g_delta[6 * (size_t)i + k] = sc.has_delta2 ? dd2[k] : 0.0f;
        a.g_delta[6 * (size_t)i + 3 + k] = sc.has_delta3 ? dd3[k] : 0.0f;
      }
    }
    if (a.g_attr) {
#pragma unroll
      for (int l = 0; l < 3; ++l)
#pragma unroll
        for (int k = 0; k < 8; ++k) a.g_attr[((size_t)l * sc.N + i) * 8 + k] = lev[l][k];
    }
#pragma unroll
    for (int k = 0; k < 3; ++k) {
      cl13[4 * k] = dmu_all[k] * g0.x + dA[4 * k]; cl13[4 * k + 1] = dmu_all[k] * g0.y + dA[4 * k + 1];
      cl13[4 * k + 2] = dmu_all[k] * g0.z + dA[4 * k + 2]; cl13[4 * k + 3] = dmu_all[k];
    }
    cl13[12] = drho[0] * acc[0] + drho[1] * acc[1] + drho[2] * acc[2];
  }
  __syncthreads();
  {
    const size_t i0 = (size_t)blockIdx.x * kPb4Threads;
    const int rows = sc.N - (int)i0 < kPb4Threads ? sc.N - (int)i0 : kPb4Threads;
    for (int f = threadIdx.x; f < rows * 3 * K; f += kPb4Threads) {
      const int r = f / (3 * K), col = f - r * (3 * K);
      a.g_shb[i0 * 3 * K + f] = s_rows[0][r * kRow + col];
      a.g_shr[i0 * 3 * K + f] = s_rows[1][r * kRow + col];
      if (a.g_dsh) {
#pragma unroll
        for (int l = 0; l < 3; ++l) a.g_dsh[((size_t)l * sc.N + i0) * 3 * K + f] = s_rows[2 + l][r * kRow + col];
      }
    }
  }
  const int c0 = __shfl_sync(0xffffffffu, c, 0);
  if (__all_sync(0xffffffffu, c == c0)) {
    if (c0 < 0) return;
#pragma unroll
    for (int k = 0; k < 13; ++k) {
      float v = cl13[k];
#pragma unroll
      for (int off = 16; off > 0; off >>= 1) v += __shfl_xor_sync(0xffffffffu, v, off);
      if (lane == 0 && v != 0.0f) atomicAdd(a.g_cluster + 13 * (size_t)c0 + k, v);
    }
  } else if (live) {
#pragma unroll
    for (int k = 0; k < 13; ++k)
      if (cl13[k] != 0.0f) atomicAdd(a.g_cluster + 13 * (size_t)c + k, cl13[k]);
  }
}

void launch_project_backward4(const DeviceScene& sc, const FrameParams& fp, const float* grad_rec, float* g_gauss,
                              float* g_shb, float* g_shr, float* g_cluster, float* g_delta, float* g_attr, float* g_dsh,
                              cudaStream_t st) {
  cudaMemsetAsync(g_cluster, 0, sizeof(float) * 13 * (size_t)sc.C, st);
  if (sc.N == 0) return;
  // a scene without that kind of refinement has zero gradient for it
  if (g_attr && !sc.g1v) { cudaMemsetAsync(g_attr, 0, sizeof(float) * 24 * (size_t)sc.N, st); g_attr = nullptr; }
  if (g_dsh && !sc.d_sh) { cudaMemsetAsync(g_dsh, 0, sizeof(float) * 9 * (size_t)sc.K * (size_t)sc.N, st); g_dsh = nullptr; }
  Pb4Args a{grad_rec, g_gauss, g_shb, g_shr, g_cluster, g_delta, g_attr, g_dsh};
  dim3 grid((sc.N + kPb4Threads - 1) / kPb4Threads), block(kPb4Threads);
  switch (sc.K) {
    case 1: k_project_backward4<1><<<grid, block, 0, st>>>(sc, fp, a); break;
    case 4: k_project_backward4<4><<<grid, block, 0, st>>>(sc, fp, a); break;
    case 9: k_project_backward4<9><<<grid, block, 0, st>>>(sc, fp, a); break;
    default: k_project_backward4<16><<<grid, block, 0, st>>>(sc, fp, a); break;
  }
  count_launches(1);
}


void launch_project_backward(const DeviceScene& sc, const FrameParams& fp, const float* grad_rec, float* g_gauss,
                             float* g_shb, float* g_shr, float* g_cluster, cudaStream_t st) {
  cudaMemsetAsync(g_cluster, 0, sizeof(float) * 13 * (size_t)sc.C, st);
  if (sc.N == 0) return;
  PbArgs a{grad_rec, g_gauss, g_shb, g_shr, g_cluster};
  dim3 grid((sc.N + kPbThreads - 1) / kPbThreads), block(kPbThreads);
  switch (sc.K) {
    case 1: k_project_backward<1><<<grid, block, 0, st>>>(sc, fp, a); break;
    case 4: k_project_backward<4><<<grid, block, 0, st>>>(sc, fp, a); break;
    case 9: k_project_backward<9><<<grid, block, 0, st>>>(sc, fp, a); break;
    default: k_project_backward<16><<<grid, block, 0, st>>>(sc, fp, a); break;
  }
  count_launches(1);
}

}  // namespace gsr
