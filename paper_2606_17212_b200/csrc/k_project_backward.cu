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
                                                 float* shb_row, float* shr_row) {
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
      const float vb[4] = {b4.x, b4.y, b4.z, b4.w};
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
        const float vb[4] = {b4.x, b4.y, b4.z, b4.w};
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
