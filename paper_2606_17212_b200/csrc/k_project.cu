// k_project.cu — stages a0..a2 of the hot path:
//   K0  closure / validation of the delivered-depth matrix (north_star (1))
//   K1  per-variant deformation (Eq. (1)) + EWA projection + SH colour
//
// Variant dedup: for a fixed (camera, t) a Gaussian has at most TWO distinct
// geometries over all B states — v=0 without the motion residual (cluster depth 0, only level-0
// Gaussians can be present then) and v=1 with it (depth >= 1) — and two colours for v=1 (with the
// level-3 SH residual iff depth == 3).  They are projected ONCE per frame instead of B times.
//
// Every quantity that feeds an integer decision is computed with explicitly rounded binary32
// intrinsics in the one operation order written in DESIGN.md §3.2/§3.3, so that the results are
// bit-identical to any other IEEE implementation of the same written order (never contracted,
// independent of -fmad / --use_fast_math).
#include "gsr_internal.h"

namespace gsr {

// ------------------------------------------------------------------------------------------------
// K0: copy levels -> ws.depth, flag anything outside -1..3 (clamped to -1 so that rendering stays defined)
__global__ void k_validate_levels(const int8_t* __restrict__ levels, int64_t n, int8_t* __restrict__ depth,
                                  WsHeader* hdr) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  int d = levels[i];
  if (d < -1 || d > 3) {
    atomicMin(&hdr->status, GSR_E_INVALID_LEVEL);  // INVALID_LEVEL (-2) wins over OK, loses to nothing above it
    d = -1;
  }
  depth[i] = (int8_t)d;
}

// also writes row B of ws.depth: the full state (every cluster at depth 3), the reference of §3.6
__global__ void k_init_header(WsHeader* hdr, int8_t* full_row, int32_t B, int32_t C, int32_t N, int32_t W,
                              int32_t H, int32_t TX, int32_t TY, long long cap) {
  for (int c = threadIdx.x; c < C; c += blockDim.x) full_row[c] = 3;
  if (threadIdx.x != 0) return;
  hdr->status = GSR_OK;
  hdr->B = B; hdr->C = C; hdr->N = N; hdr->W = W; hdr->H = H; hdr->TX = TX; hdr->TY = TY;
  hdr->total_keys = 0; hdr->n_keys = 0; hdr->key_capacity = cap;
}

void launch_validate_levels(const int8_t* levels, int32_t B, int32_t C, Workspace& ws, cudaStream_t st) {
  int64_t n = (int64_t)B * C;
  if (n == 0) return;
  k_validate_levels<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(levels, n, ws.depth, ws.hdr);
  count_launches(1);
}

// dependency closure of raw 4-bit delivery masks: depth = (#trailing one bits) - 1
__global__ void k_close_levels(const uint8_t* __restrict__ mask, int64_t n, int8_t* __restrict__ depth,
                               uint8_t* __restrict__ closure) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  unsigned m = mask[i] & 0xFu;
  int run = __ffs(~m) - 1;  // index of the lowest zero bit = number of trailing ones (m has only 4 bits)
  depth[i] = (int8_t)(run - 1);
  if (closure) closure[i] = (uint8_t)((1u << run) - 1u);
}

void launch_close_levels(const uint8_t* mask, int64_t n, int8_t* depth, uint8_t* closure, cudaStream_t st) {
  if (n == 0) return;
  k_close_levels<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(mask, n, depth, closure);
  count_launches(1);
}

// ------------------------------------------------------------------------------------------------
// K1 helpers
struct Proj {
  float mx, my, qa, qb, qc;
  float hx, hy;  // conservative half-extents (pixels) of the region where the cut q <= tau can pass
  int radius;
  int tx0, ty0, tx1, ty1;
  uint32_t depth_bits;
  uint32_t count;  // 0 = culled
};

__device__ __forceinline__ float clampf_rn(float v, float lo, float hi) { return fminf(hi, fmaxf(lo, v)); }

// EWA projection of a world-space mean `mu` with 3-D covariance S (xx xy xz yy yz zz).
__device__ __forceinline__ Proj project_variant(const FrameParams& fp, const float mu[3], const float S6[6],
                                                const float tau) {
  Proj o;
  o.count = 0; o.radius = 0; o.tx0 = o.ty0 = o.tx1 = o.ty1 = 0; o.depth_bits = 0;
  o.mx = o.my = o.qa = o.qb = o.qc = 0.f;
  o.hx = o.hy = 0.f;
  const float* Rw = fp.R;
  float pc[3];
#pragma unroll
  for (int k = 0; k < 3; ++k)
    pc[k] = __fmaf_rn(Rw[3 * k + 0], mu[0], __fmaf_rn(Rw[3 * k + 1], mu[1], __fmaf_rn(Rw[3 * k + 2], mu[2], fp.t[k])));
  float z = pc[2];
  if (!(z > fp.znear)) return o;
  float rz = __fdiv_rn(1.0f, z);
  float txz = __fmul_rn(pc[0], rz);
  float tyz = __fmul_rn(pc[1], rz);
  float limx = __fmul_rn(__fdiv_rn(__fmul_rn(0.5f, (float)fp.W), fp.fx), 1.3f);
  float limy = __fmul_rn(__fdiv_rn(__fmul_rn(0.5f, (float)fp.H), fp.fy), 1.3f);
  float xt = __fmul_rn(clampf_rn(txz, -limx, limx), z);
  float yt = __fmul_rn(clampf_rn(tyz, -limy, limy), z);
  float J00 = __fmul_rn(fp.fx, rz);
  float J02 = -__fmul_rn(__fmul_rn(__fmul_rn(fp.fx, xt), rz), rz);
  float J11 = __fmul_rn(fp.fy, rz);
  float J12 = -__fmul_rn(__fmul_rn(__fmul_rn(fp.fy, yt), rz), rz);
  float M0[3], M1[3];
#pragma unroll
  for (int k = 0; k < 3; ++k) {
    M0[k] = __fmaf_rn(J02, Rw[6 + k], __fmul_rn(J00, Rw[0 + k]));
    M1[k] = __fmaf_rn(J12, Rw[6 + k], __fmul_rn(J11, Rw[3 + k]));
  }
  const float S[9] = {S6[0], S6[1], S6[2], S6[1], S6[3], S6[4], S6[2], S6[4], S6[5]};
  float v0[3], v1[3];
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    v0[a] = __fmaf_rn(S[3 * a + 2], M0[2], __fmaf_rn(S[3 * a + 1], M0[1], __fmul_rn(S[3 * a + 0], M0[0])));
    v1[a] = __fmaf_rn(S[3 * a + 2], M1[2], __fmaf_rn(S[3 * a + 1], M1[1], __fmul_rn(S[3 * a + 0], M1[0])));
  }
  float s00 = __fmaf_rn(M0[2], v0[2], __fmaf_rn(M0[1], v0[1], __fmul_rn(M0[0], v0[0])));
  float s01 = __fmaf_rn(M0[2], v1[2], __fmaf_rn(M0[1], v1[1], __fmul_rn(M0[0], v1[0])));
  float s11 = __fmaf_rn(M1[2], v1[2], __fmaf_rn(M1[1], v1[1], __fmul_rn(M1[0], v1[0])));
  float a = __fadd_rn(s00, 0.3f), b = s01, c = __fadd_rn(s11, 0.3f);
  float det = __fmaf_rn(a, c, -__fmul_rn(b, b));
  if (!(det > 0.0f)) return o;
  float rdet = __fdiv_rn(1.0f, det);
  float conic_a = __fmul_rn(c, rdet), conic_b = -__fmul_rn(b, rdet), conic_c = __fmul_rn(a, rdet);
  float mid = __fmul_rn(0.5f, __fadd_rn(a, c));
  float disc = fmaxf(0.1f, __fmaf_rn(mid, mid, -det));
  float lam = __fadd_rn(mid, __fsqrt_rn(disc));
  float rad = ceilf(__fmul_rn(3.0f, __fsqrt_rn(lam)));
  float mx = __fmaf_rn(fp.fx, txz, fp.cx);
  float my = __fmaf_rn(fp.fy, tyz, fp.cy);
  float TXf = (float)fp.TX, TYf = (float)fp.TY;
  int tx0 = (int)clampf_rn(floorf(__fmul_rn(__fsub_rn(mx, rad), 0.0625f)), 0.0f, TXf);
  int tx1 = (int)clampf_rn(floorf(__fmul_rn(__fadd_rn(__fadd_rn(mx, rad), 15.0f), 0.0625f)), 0.0f, TXf);
  int ty0 = (int)clampf_rn(floorf(__fmul_rn(__fsub_rn(my, rad), 0.0625f)), 0.0f, TYf);
  int ty1 = (int)clampf_rn(floorf(__fmul_rn(__fadd_rn(__fadd_rn(my, rad), 15.0f), 0.0625f)), 0.0f, TYf);
  o.mx = mx; o.my = my;
  o.qa = __fmul_rn(0.5f, conic_a); o.qb = conic_b; o.qc = __fmul_rn(0.5f, conic_c);
  {
    // Sub-tile culling bound: {q <= tau} is the ellipse x^T Sigma'^-1 x <= 2 tau, whose
    // half-extents are sqrt(2 tau a), sqrt(2 tau c).  The kernel evaluates q in fp32 from the ROUNDED
    // conic, so the bound is inflated by m = 8e-6 kappa + 1e-3, kappa = a c / det >= 1 (conditioning of
    // the form: bounds both the conic rounding and the cancellation in q, each < 3e-6 kappa), and tau by
    // +1e-2 (covers tau <= 0 and q rounding to a tiny negative).  Continuous, never feeds a list decision.
    const float kappa = a * c * rdet;
    const float m = 1.0f + fminf(1.0f, 8e-6f * kappa + 1e-3f);
    const float t2 = 2.0f * (fmaxf(tau, 0.0f) + 1e-2f);
    o.hx = sqrtf(t2 * a) * m + 1e-3f;
    o.hy = sqrtf(t2 * c) * m + 1e-3f;
  }
  o.radius = (int)rad;
  if (tx1 <= tx0 || ty1 <= ty0) return o;
  o.tx0 = tx0; o.ty0 = ty0; o.tx1 = tx1; o.ty1 = ty1;
  o.count = (uint32_t)((tx1 - tx0) * (ty1 - ty0));
  o.depth_bits = __float_as_uint(z);
  return o;
}

// real orthonormal SH basis to degree 3 at unit direction (x,y,z) — DESIGN.md §3.3 (colour); the
// constants are the textbook ones, written as decimals here.
template <int K>
__device__ __forceinline__ void sh_eval(float x, float y, float z, float* Y) {
  Y[0] = 0.28209479177387814f;
  if (K > 1) {
    Y[1] = 0.4886025119029199f * y;
    Y[2] = 0.4886025119029199f * z;
    Y[3] = 0.4886025119029199f * x;
  }
  if (K > 4) {
    float xx = x * x, yy = y * y, zz = z * z;
    Y[4] = 1.0925484305920792f * x * y;
    Y[5] = 1.0925484305920792f * y * z;
    Y[6] = 0.31539156525252005f * (3.0f * zz - 1.0f);
    Y[7] = 1.0925484305920792f * x * z;
    Y[8] = 0.5462742152960396f * (xx - yy);
    if (K > 9) {
      Y[9] = 0.5900435899266435f * y * (3.0f * xx - yy);
      Y[10] = 2.890611442640554f * x * y * z;
      Y[11] = 0.4570457994644658f * y * (5.0f * zz - 1.0f);
      Y[12] = 0.3731763325901154f * (5.0f * zz * z - 3.0f * z);
      Y[13] = 0.4570457994644658f * x * (5.0f * zz - 1.0f);
      Y[14] = 1.445305721320277f * (xx - yy) * z;
      Y[15] = 0.5900435899266435f * x * (xx - 3.0f * yy);
    }
  }
}

template <int K>
__device__ __forceinline__ void sh_dir(const FrameParams& fp, const float mu[3], float* Y) {
  float dx = mu[0] - fp.cam_centre[0], dy = mu[1] - fp.cam_centre[1], dz = mu[2] - fp.cam_centre[2];
  float inv = rsqrtf(dx * dx + dy * dy + dz * dz);
  sh_eval<K>(dx * inv, dy * inv, dz * inv, Y);
}

// Also the first step of the binning (k_sort.cu): one increment per tile of the record's rectangle.  The
// increments are fire-and-forget reductions that overlap the kernel's own memory latency.
// And the packed 64-byte record the compositor stages (k_composite_q.cu):
//   {m_x, m_y, A, B} {Cq, tau, o, meta} {rgb - bg, 0} {rgb with SH residual - bg, 0}
__device__ __forceinline__ void store_record(Workspace& ws, const FrameParams& fp, uint32_t rid, const Proj& p,
                                             float opac, float tau, uint32_t meta, const float* c0, const float* c1) {
  const int TX = fp.TX;
  float4* rec = ws.rec + 4 * (size_t)rid;
  rec[0] = make_float4(p.mx, p.my, p.qa, p.qb);
  rec[1] = make_float4(p.qc, tau, opac, __uint_as_float(meta));
  rec[2] = make_float4(__fsub_rn(c0[0], fp.bg[0]), __fsub_rn(c0[1], fp.bg[1]), __fsub_rn(c0[2], fp.bg[2]), 0.0f);
  rec[3] = make_float4(__fsub_rn(c1[0], fp.bg[0]), __fsub_rn(c1[1], fp.bg[1]), __fsub_rn(c1[2], fp.bg[2]), 0.0f);
  ws.r0[rid] = make_float4(p.mx, p.my, p.qa, p.qb);
  ws.r1[rid] = make_float4(p.qc, opac, tau, __uint_as_float(meta));
  ws.rc0[rid] = make_float4(c0[0], c0[1], c0[2], p.hx);
  ws.rc1[rid] = make_float4(c1[0], c1[1], c1[2], p.hy);
  ws.radius[rid] = p.radius;
  ws.rect[rid] = make_uint2((uint32_t)p.tx0 | ((uint32_t)p.ty0 << 16), (uint32_t)p.tx1 | ((uint32_t)p.ty1 << 16));
  ws.depth_bits[rid] = p.depth_bits;
  ws.count[rid] = p.count;
  if (p.count != 0)
    for (int ty = p.ty0; ty < p.ty1; ++ty)
      for (int tx = p.tx0; tx < p.tx1; ++tx) atomicAdd(ws.tile_cursor + ty * TX + tx, 1u);
}

// reading I4 (optional): Sigma_t = L Sigma L^T, L = the 3x3 part of A_c(t); binary32 in the written order of
// Mm = L S (row a, column b), then Sigma_t[a][b] = Mm[a] . L[b]
__device__ __forceinline__ void push_forward_cov(const float* A, const float* S6, float* out6) {
  const float Sf[9] = {S6[0], S6[1], S6[2], S6[1], S6[3], S6[4], S6[2], S6[4], S6[5]};
  float Mm[9];
#pragma unroll
  for (int a = 0; a < 3; ++a)
#pragma unroll
    for (int b = 0; b < 3; ++b)
      Mm[3 * a + b] = __fmaf_rn(A[4 * a + 2], Sf[6 + b], __fmaf_rn(A[4 * a + 1], Sf[3 + b], __fmul_rn(A[4 * a + 0], Sf[b])));
  int o = 0;
#pragma unroll
  for (int a = 0; a < 3; ++a)
#pragma unroll
    for (int b = a; b < 3; ++b)
      out6[o++] = __fmaf_rn(Mm[3 * a + 2], A[4 * b + 2], __fmaf_rn(Mm[3 * a + 1], A[4 * b + 1], __fmul_rn(Mm[3 * a + 0], A[4 * b + 0])));
}

// K1: one thread per Gaussian; record id = 2*i + v.
template <int K>
__global__ void __launch_bounds__(128) k_project(DeviceScene sc, FrameParams fp, Workspace ws) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= sc.N) return;
  const float4 g0 = __ldg(sc.g0 + i), g1 = __ldg(sc.g1 + i), g2 = __ldg(sc.g2 + i);
  const uint32_t bits = __float_as_uint(g2.w);
  const int c = (int)(bits >> 2), lvl = (int)(bits & 3u);
  const float S6[6] = {g1.x, g1.y, g1.z, g2.x, g2.y, g2.z};
  const float opac = g0.w, tau = g1.w;

  // ---- Eq. (1): A = A0 + t A1 ; p = A [mu_bar; 1] ; residual = s_c * sum_r b_r q_r
  const float* A0 = sc.A0 + 12 * c;
  const float* A1 = sc.A1 + 12 * c;
  float A[12];
#pragma unroll
  for (int k = 0; k < 12; ++k) A[k] = __fmaf_rn(fp.time, __ldg(A1 + k), __ldg(A0 + k));
  float p[3];
#pragma unroll
  for (int k = 0; k < 3; ++k)
    p[k] = __fmaf_rn(A[4 * k + 0], g0.x, __fmaf_rn(A[4 * k + 1], g0.y, __fmaf_rn(A[4 * k + 2], g0.z, A[4 * k + 3])));
  float acc[3] = {0.f, 0.f, 0.f};
  {
    uint32_t w = 0;
    for (int r = 0; r < sc.R; ++r) {
#pragma unroll
      for (int k = 0; k < 3; ++k) {
        int byte = r * 3 + k;
        if ((byte & 3) == 0) w = __ldg(sc.qw + (size_t)(byte >> 2) * sc.N + i);
        int q = (int)(int8_t)((w >> ((byte & 3) * 8)) & 0xFFu);
        acc[k] = __fmaf_rn(fp.basis[r], (float)q, acc[k]);
      }
    }
  }
  const float s_c = __ldg(sc.mscale + c);
  float muB[3];
#pragma unroll
  for (int k = 0; k < 3; ++k) muB[k] = __fmaf_rn(s_c, acc[k], p[k]);

  // ---- EWA projection of both geometries
  float St[6];
  const float* Sp = S6;
  if (sc.affine_cov) { push_forward_cov(A, S6, St); Sp = St; }
  Proj pa{};  // absent variant: all fields zero (gsr_debug_projection exports them), count = 0 = culled
  if (lvl == 0) pa = project_variant(fp, p, Sp, tau);
  Proj pb = project_variant(fp, muB, Sp, tau);

  // ---- colour (continuous; fp32): rgb = max(0, 0.5 + sum_j Y_j(dir) * coef_j)
  float cA[3] = {0.f, 0.f, 0.f}, cB0[3] = {0.f, 0.f, 0.f}, cB1[3] = {0.f, 0.f, 0.f};
  const bool needA = (lvl == 0) && pa.count > 0, needB = pb.count > 0;
  if (needA || needB) {
    float YA[K], YB[K];
    sh_dir<K>(fp, p, YA);
    sh_dir<K>(fp, muB, YB);
    float sa[3] = {0.5f, 0.5f, 0.5f}, sb0[3] = {0.5f, 0.5f, 0.5f}, sb1[3] = {0.f, 0.f, 0.f};
    constexpr int n4 = (3 * K + 3) / 4;
#pragma unroll
    for (int w4 = 0; w4 < n4; ++w4) {
      const float4 cb = __ldg(sc.sh_base + (size_t)w4 * sc.N + i);
      const float4 cr = __ldg(sc.sh_res + (size_t)w4 * sc.N + i);
      const float vb[4] = {cb.x, cb.y, cb.z, cb.w}, vr[4] = {cr.x, cr.y, cr.z, cr.w};
#pragma unroll
      for (int e = 0; e < 4; ++e) {
        const int flat = w4 * 4 + e;
        if (flat < 3 * K) {
          const int j = flat / 3, ch = flat % 3;
          sa[ch] = fmaf(YA[j], vb[e], sa[ch]);
          sb0[ch] = fmaf(YB[j], vb[e], sb0[ch]);
          sb1[ch] = fmaf(YB[j], vr[e], sb1[ch]);
        }
      }
    }
#pragma unroll
    for (int ch = 0; ch < 3; ++ch) {
      cA[ch] = fmaxf(0.f, sa[ch]);
      cB0[ch] = fmaxf(0.f, sb0[ch]);
      cB1[ch] = fmaxf(0.f, sb0[ch] + sb1[ch]);
    }
  }
  // record class: 0 = variant A (depth == 0), 1 + lvl = variant B of a level-lvl Gaussian
  store_record(ws, fp, 2u * i + 0u, pa, opac, tau, (uint32_t)c | (0u << 16), cA, cA);
  store_record(ws, fp, 2u * i + 1u, pb, opac, tau, (uint32_t)c | ((uint32_t)(1 + lvl) << 16), cB0, cB1);
}

// K1 with the position residual levels of Eq. (1) (reading I1): a Gaussian has one geometry per
// delivered depth d = 0..3 — p (affine only), p + motion residual, + delta2, + delta3 — and variant v is present
// exactly in the states whose cluster depth is v (v = 3: depth 3, with the SH residual colour).  A level-l
// Gaussian only has the variants v >= l.  Record id = 4*i + v, record class 16 + v.
template <int K>
__global__ void __launch_bounds__(128) k_project4(DeviceScene sc, FrameParams fp, Workspace ws) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= sc.N) return;
  const float4 g0 = __ldg(sc.g0 + i), g1 = __ldg(sc.g1 + i), g2 = __ldg(sc.g2 + i);
  const uint32_t bits = __float_as_uint(g2.w);
  const int c = (int)(bits >> 2), lvl = (int)(bits & 3u);
  const float S6[6] = {g1.x, g1.y, g1.z, g2.x, g2.y, g2.z};
  const float opac = g0.w, tau = g1.w;
  const float* A0 = sc.A0 + 12 * c;
  const float* A1 = sc.A1 + 12 * c;
  float A[12];
#pragma unroll
  for (int k = 0; k < 12; ++k) A[k] = __fmaf_rn(fp.time, __ldg(A1 + k), __ldg(A0 + k));
  float mu[4][3];
#pragma unroll
  for (int k = 0; k < 3; ++k)
    mu[0][k] = __fmaf_rn(A[4 * k + 0], g0.x, __fmaf_rn(A[4 * k + 1], g0.y, __fmaf_rn(A[4 * k + 2], g0.z, A[4 * k + 3])));
  float acc[3] = {0.f, 0.f, 0.f};
  {
    uint32_t w = 0;
    for (int r = 0; r < sc.R; ++r) {
#pragma unroll
      for (int k = 0; k < 3; ++k) {
        int byte = r * 3 + k;
        if ((byte & 3) == 0) w = __ldg(sc.qw + (size_t)(byte >> 2) * sc.N + i);
        int q = (int)(int8_t)((w >> ((byte & 3) * 8)) & 0xFFu);
        acc[k] = __fmaf_rn(fp.basis[r], (float)q, acc[k]);
      }
    }
  }
  const float s_c = __ldg(sc.mscale + c);
#pragma unroll
  for (int k = 0; k < 3; ++k) {
    mu[1][k] = __fmaf_rn(s_c, acc[k], mu[0][k]);
    mu[2][k] = __fadd_rn(mu[1][k], __ldg(sc.delta + (size_t)k * sc.N + i));
    mu[3][k] = __fadd_rn(mu[2][k], __ldg(sc.delta + (size_t)(3 + k) * sc.N + i));
  }
  Proj pr[4];
  float opv[4], tauv[4];
  bool any = false;
#pragma unroll
  for (int v = 0; v < 4; ++v) {
    pr[v] = Proj{};  // absent variant: all fields zero, count = 0 = culled
    opv[v] = opac; tauv[v] = tau;
    if (v >= lvl) {
      if (sc.g1v) {  // scale / rotation / opacity refinements (reading I2): attributes of delivered depth v
        const float4 h1 = __ldg(sc.g1v + (size_t)v * sc.N + i), h2 = __ldg(sc.g2v + (size_t)v * sc.N + i);
        float Sv[6] = {h1.x, h1.y, h1.z, h2.x, h2.y, h2.z};
        if (sc.affine_cov) { float Sx[6]; push_forward_cov(A, Sv, Sx); for (int k = 0; k < 6; ++k) Sv[k] = Sx[k]; }
        opv[v] = __ldg(sc.opv + (size_t)v * sc.N + i);
        tauv[v] = h1.w;
        pr[v] = project_variant(fp, mu[v], Sv, tauv[v]);
      } else {
        float St[6];
        const float* Sp = S6;
        if (sc.affine_cov) { push_forward_cov(A, S6, St); Sp = St; }
        pr[v] = project_variant(fp, mu[v], Sp, tau);
      }
    }
    any |= pr[v].count > 0;
  }
  float col[4][3] = {{0.f, 0.f, 0.f}, {0.f, 0.f, 0.f}, {0.f, 0.f, 0.f}, {0.f, 0.f, 0.f}};
  if (any) {
    constexpr int n4 = (3 * K + 3) / 4;
#pragma unroll
    for (int v = 0; v < 4; ++v) {
      if (pr[v].count == 0) continue;
      float Y[K];
      sh_dir<K>(fp, mu[v], Y);
      float sb[3] = {0.5f, 0.5f, 0.5f}, sr[3] = {0.f, 0.f, 0.f};
#pragma unroll
      for (int w4 = 0; w4 < n4; ++w4) {
        float4 cb = __ldg(sc.sh_base + (size_t)w4 * sc.N + i);
        const float4 cr = __ldg(sc.sh_res + (size_t)w4 * sc.N + i);
        if (sc.d_sh) {  // colour refinements of the delivered levels 1..v (reading I3)
          for (int l = 0; l < v; ++l) {
            const float4 dl = __ldg(sc.d_sh + ((size_t)l * n4 + w4) * sc.N + i);
            cb.x += dl.x; cb.y += dl.y; cb.z += dl.z; cb.w += dl.w;
          }
        }
        const float vb[4] = {cb.x, cb.y, cb.z, cb.w}, vr[4] = {cr.x, cr.y, cr.z, cr.w};
#pragma unroll
        for (int e = 0; e < 4; ++e) {
          const int flat = w4 * 4 + e;
          if (flat < 3 * K) {
            const int j = flat / 3, ch = flat % 3;
            sb[ch] = fmaf(Y[j], vb[e], sb[ch]);
            sr[ch] = fmaf(Y[j], vr[e], sr[ch]);
          }
        }
      }
#pragma unroll
      for (int ch = 0; ch < 3; ++ch) col[v][ch] = fmaxf(0.f, v == 3 ? sb[ch] + sr[ch] : sb[ch]);
    }
  }
#pragma unroll
  for (int v = 0; v < 4; ++v)
    store_record(ws, fp, 4u * i + (uint32_t)v, pr[v], opv[v], tauv[v], (uint32_t)c | ((uint32_t)(16 + v) << 16), col[v], col[v]);
}

void launch_project(const DeviceScene& sc, const FrameParams& fp, Workspace& ws, cudaStream_t st) {
  cudaMemsetAsync(ws.tile_cursor, 0, sizeof(uint32_t) * (size_t)fp.TX * fp.TY, st);  // keys per tile, counted below
  if (sc.N == 0) return;
  dim3 grid((sc.N + 127) / 128), block(128);
  if (sc.V == 4) {
    switch (sc.K) {
      case 1: k_project4<1><<<grid, block, 0, st>>>(sc, fp, ws); break;
      case 4: k_project4<4><<<grid, block, 0, st>>>(sc, fp, ws); break;
      case 9: k_project4<9><<<grid, block, 0, st>>>(sc, fp, ws); break;
      default: k_project4<16><<<grid, block, 0, st>>>(sc, fp, ws); break;
    }
    count_launches(1);
    return;
  }
  switch (sc.K) {
    case 1: k_project<1><<<grid, block, 0, st>>>(sc, fp, ws); break;
    case 4: k_project<4><<<grid, block, 0, st>>>(sc, fp, ws); break;
    case 9: k_project<9><<<grid, block, 0, st>>>(sc, fp, ws); break;
    default: k_project<16><<<grid, block, 0, st>>>(sc, fp, ws); break;
  }
  count_launches(1);
}

void launch_init_header(Workspace& ws, int32_t B, int32_t C, int32_t N, const FrameParams& fp, long long cap,
                        cudaStream_t st) {
  k_init_header<<<1, 256, 0, st>>>(ws.hdr, ws.depth + (size_t)B * C, B, C, N, fp.W, fp.H, fp.TX, fp.TY, cap);
  count_launches(1);
}

}  // namespace gsr
