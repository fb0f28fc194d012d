/*
 * gsr_oracle.c — the CPU ORACLE for the batched counterfactual-state Gaussian renderer.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  It is a plain, slow, obviously-correct CPU
 * restatement of what the hot path computes.  It shares no code, header, table or constant with
 * the CUDA path under paper_2606_17212_b200/csrc/.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may build, load or call it.
 *
 * What it follows (PAPER.md = /root/reference/PAPER.md; DESIGN.md §3 = the written spec):
 *   O-0 activation at load ........ DESIGN.md §3.0      (exp / sigmoid / quaternion -> Sigma; double -> fp32 once)
 *   O-1 dependency closure ........ PAPER.md:64,164,185 ("usable only when all chunks in its
 *                                   dependency closure are usable"), BASELINE.json configs[0]
 *   O-2 deformation ............... PAPER.md:46-50, Eq. (1): mu = A_{c,t} mu_bar + sum_r b_{t,r} q_{i,r} + delta^(2) + delta^(3)
 *   O-3 EWA projection ............ PAPER.md:140 delegates to a splatting library and prints nothing;
 *                                   the definition is the standard EWA one fixed by BASELINE.json
 *                                   north_star (2) and DESIGN.md §3.3 (every constant is a listed reading)
 *   O-4 order ..................... north_star (3): (state, tile, depth, gaussian-index), keys unique
 *   O-5 pixel ..................... north_star (4): per-pixel brute force over ALL depth-sorted Gaussians,
 *                                   front-to-back alpha compositing with early termination
 *   O-6 distortion ................ north_star (5): MSE / PSNR against the full-state render
 *   O-7 utility ................... PAPER.md:80-88, Eq. (3) and Eq. (4) (alpha=0.25, beta=0.05, Q_0.1)
 *   O-8 backward of O-5 ........... PAPER.md:64-76 (the objective is a function of the rendered images): the
 *                                   gradient of a linear functional of one state's image with respect to the
 *                                   2-D quantities O-5 reads; the chain rule of O-5 written out, decisions fixed
 *                                   (pins: tests/test_backward_pins.py — finite differences of O-5, closed form)
 *   O-9 backward of O-0/O-2/O-3 ... the same chain one step further back: from the gradient with respect to the
 *                                   2-D quantities of a Gaussian in one state (O-8's output) to the gradient with
 *                                   respect to the scene's own parameters (mean, motion residual, log-scale,
 *                                   quaternion, opacity logit, SH coefficients, cluster affine, s_c); the chain
 *                                   rule of DESIGN.md §3.0-§3.3 written out in double, decisions fixed
 *                                   (pins: tests/test_projection_backward_pins.py — finite differences of
 *                                   O-0/O-2/O-3, closed forms, invariants)
 *
 * Precision split.  Quantities that feed an INTEGER decision (deformed mean,
 * camera-space point, 2-D covariance, conic, radius, tile rectangle, depth bits, the quadratic
 * form q and the test q > tau) are computed in IEEE binary32 with ONE written operation order
 * (fmaf explicit, build with -ffp-contract=off) so that another implementation can match them bit
 * for bit.  Continuous quantities (SH colour, exp(-q), alpha, T, C, SSE) are computed in double
 * from those fp32 values.
 *
 * Parity pins: tests/test_oracle_pins.py (P1..P16 of SURVEY.md §8(c)).  Unpinned: parity with the
 * PAPER's own pixels/utilities (needs its trained scenes + renderer, which are not available) —
 * "parity unpinned" for that item only; every function below has at least one pin.
 *
 * Build: gcc -O2 -ffp-contract=off -fno-fast-math -mfma -fopenmp -shared -fPIC (see oracle/oracle.py).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#ifdef _OPENMP
#include <omp.h>
#endif

#define TILE 16

/* ------------------------------------------------------------------------------------------ */
/* types                                                                                       */
/* ------------------------------------------------------------------------------------------ */

typedef struct {
  int32_t C, N, K, R; /* K = (sh_degree+1)^2 coefficients per channel */
  const int32_t* group_off; /* [4C+1]  Gaussians sorted by (cluster, level) */
  const float* mean;        /* [N,3]   canonical mu_bar                      */
  const float* cov3d;       /* [N,6]   activated: xx xy xz yy yz zz          */
  const float* opacity;     /* [N]     activated sigmoid                     */
  const float* tau;         /* [N]     ln(255 * opacity)                     */
  const float* sh_base;     /* [N,K,3]                                       */
  const float* sh_res;      /* [N,K,3] level-3 payload                       */
  const int8_t* motion_q;   /* [N,R,3] level-1 payload                       */
  const float* A0;          /* [C,3,4] */
  const float* A1;          /* [C,3,4] */
  const float* motion_scale; /* [C]    */
  const float* delta2;      /* [N,3] level-2 position residual delta^(2) of Eq. (1), or NULL (= 0) */
  const float* delta3;      /* [N,3] level-3 position residual delta^(3) of Eq. (1), or NULL (= 0) */
  /* per-depth activated attributes of scenes with scale / rotation / opacity refinements (PAPER.md:50,
   * DESIGN.md reading I2), or NULL: [4][N,6], [4][N], [4][N] for delivered depth 0..3 */
  const float* cov3d_lv;
  const float* opacity_lv;
  const float* tau_lv;
  const float* d_sh;        /* [3][N,K,3] per-level colour residuals (levels 1..3; reading I3), or NULL */
  int32_t affine_cov;       /* != 0: the cluster affine also transforms the covariance (reading I4) */
  int32_t pad_;
  float background[3];
} orc_scene;

typedef struct {
  float R[9], t[3], fx, fy, cx, cy;
  int32_t W, H;
  float znear;
} orc_camera;

/* one Gaussian of one state after O-2/O-3 */
typedef struct {
  int32_t valid;       /* 1 = present in the state and not culled      */
  float mu[3];         /* deformed world position (O-2)                */
  float z;             /* camera-space depth                           */
  float mx, my;        /* 2-D mean in pixels                           */
  float qa, qb, qc;    /* A = conic_a/2, B = conic_b, Cq = conic_c/2   */
  float cov2d[3];      /* a, b, c after the +0.3 dilation              */
  int32_t radius;      /* ceil(3 sqrt(lambda_max))                     */
  int32_t rect[4];     /* tx0, ty0, tx1, ty1 (half-open, in tiles)     */
  uint32_t depth_bits; /* raw bits of z                                */
  int32_t count;       /* tiles touched                                */
  double rgb[3];       /* SH colour (continuous)                       */
  float opacity, tau;  /* activated opacity and ln(255 opacity) at this state's depth */
  float pad_[2];
} orc_proj;

/* ------------------------------------------------------------------------------------------ */
/* O-1  dependency closure                               */
/* ------------------------------------------------------------------------------------------ */

/* mask bit l = "level-l completion group of this cluster is usable".  Level l is renderable iff
 * levels 0..l are all usable, so the delivered depth is (number of trailing one bits) - 1. */
void orc_close_levels(const uint8_t* mask, int64_t n, int8_t* depth, uint8_t* closure) {
  for (int64_t i = 0; i < n; ++i) {
    int d = -1;
    for (int l = 0; l < 4; ++l) {
      if ((mask[i] >> l) & 1)
        d = l;
      else
        break;
    }
    depth[i] = (int8_t)d;
    closure[i] = (uint8_t)((1u << (d + 1)) - 1u);
  }
}

/* ------------------------------------------------------------------------------------------ */
/* O-0  activation at load — double, rounded to fp32 once                    */
/* ------------------------------------------------------------------------------------------ */

void orc_activate(int64_t N, const float* log_scale, const float* quat, const float* logit,
                  float* cov3d, float* opacity, float* tau) {
  for (int64_t i = 0; i < N; ++i) {
    double s[3];
    for (int k = 0; k < 3; ++k) s[k] = exp((double)log_scale[3 * i + k]);
    double w = quat[4 * i + 0], x = quat[4 * i + 1], y = quat[4 * i + 2], z = quat[4 * i + 3];
    double n = sqrt(w * w + x * x + y * y + z * z);
    w /= n; x /= n; y /= n; z /= n;
    double Rm[9] = {1.0 - 2.0 * (y * y + z * z), 2.0 * (x * y - w * z),       2.0 * (x * z + w * y),
                    2.0 * (x * y + w * z),       1.0 - 2.0 * (x * x + z * z), 2.0 * (y * z - w * x),
                    2.0 * (x * z - w * y),       2.0 * (y * z + w * x),       1.0 - 2.0 * (x * x + y * y)};
    double M[9]; /* M = Rm * diag(s) */
    for (int a = 0; a < 3; ++a)
      for (int k = 0; k < 3; ++k) M[3 * a + k] = Rm[3 * a + k] * s[k];
    /* Sigma = M M^T */
    int o = 0;
    for (int a = 0; a < 3; ++a)
      for (int b = a; b < 3; ++b) {
        double acc = M[3 * a + 0] * M[3 * b + 0];
        acc += M[3 * a + 1] * M[3 * b + 1];
        acc += M[3 * a + 2] * M[3 * b + 2];
        cov3d[6 * i + o++] = (float)acc;
      }
    float of = (float)(1.0 / (1.0 + exp(-(double)logit[i])));
    opacity[i] = of;
    tau[i] = (float)log(255.0 * (double)of);
  }
}

/* temporal basis b_r(t) = cos(pi r t), r = 1..R  (reading A6), double -> fp32 */
void orc_basis(float t, int32_t R, float* b) {
  for (int r = 1; r <= R; ++r) b[r - 1] = (float)cos(M_PI * (double)r * (double)t);
}

/* ------------------------------------------------------------------------------------------ */
/* real spherical harmonics to degree 3 (textbook orthonormal basis, DESIGN.md §3.3 colour)    */
/* ------------------------------------------------------------------------------------------ */

static void sh_basis(int K, double x, double y, double z, double* Y) {
  const double pi = M_PI;
  Y[0] = 0.5 * sqrt(1.0 / pi);
  if (K <= 1) return;
  double c1 = sqrt(3.0 / (4.0 * pi));
  Y[1] = c1 * y;
  Y[2] = c1 * z;
  Y[3] = c1 * x;
  if (K <= 4) return;
  Y[4] = 0.5 * sqrt(15.0 / pi) * x * y;
  Y[5] = 0.5 * sqrt(15.0 / pi) * y * z;
  Y[6] = 0.25 * sqrt(5.0 / pi) * (3.0 * z * z - 1.0);
  Y[7] = 0.5 * sqrt(15.0 / pi) * x * z;
  Y[8] = 0.25 * sqrt(15.0 / pi) * (x * x - y * y);
  if (K <= 9) return;
  Y[9] = 0.25 * sqrt(35.0 / (2.0 * pi)) * y * (3.0 * x * x - y * y);
  Y[10] = 0.5 * sqrt(105.0 / pi) * x * y * z;
  Y[11] = 0.25 * sqrt(21.0 / (2.0 * pi)) * y * (5.0 * z * z - 1.0);
  Y[12] = 0.25 * sqrt(7.0 / pi) * (5.0 * z * z * z - 3.0 * z);
  Y[13] = 0.25 * sqrt(21.0 / (2.0 * pi)) * x * (5.0 * z * z - 1.0);
  Y[14] = 0.25 * sqrt(105.0 / pi) * (x * x - y * y) * z;
  Y[15] = 0.25 * sqrt(35.0 / (2.0 * pi)) * x * (x * x - 3.0 * y * y);
}

/* exported for the orthonormality pin (P9) */
void orc_sh_basis(int32_t K, double x, double y, double z, double* Y) { sh_basis(K, x, y, z, Y); }

/* ------------------------------------------------------------------------------------------ */
/* O-2 + O-3  deformation and EWA projection of Gaussian i in a state whose cluster depth is d */
/* ------------------------------------------------------------------------------------------ */

static int level_of(const orc_scene* s, int c, int i) {
  int l = 0;
  while (l < 3 && i >= s->group_off[4 * c + l + 1]) ++l;
  return l;
}

static float clampf(float v, float lo, float hi) { return fminf(hi, fmaxf(lo, v)); }

static void project_one(const orc_scene* s, const orc_camera* cam, float t, const float* basis,
                        int c, int i, int d, orc_proj* o) {
  memset(o, 0, sizeof(*o));
  int lvl = level_of(s, c, i);
  if (d < lvl) return; /* O-1: present iff d >= level(i); d = -1 removes the whole cluster */
  o->opacity = s->opacity_lv ? s->opacity_lv[(int64_t)d * s->N + i] : s->opacity[i];
  o->tau = s->tau_lv ? s->tau_lv[(int64_t)d * s->N + i] : s->tau[i];

  /* ---- O-2 (Eq. 1): A = A0 + t A1 ; p = A [mu_bar;1] ; residual = s_c * sum_r b_r q_r ---- */
  const float* A0 = s->A0 + 12 * c;
  const float* A1 = s->A1 + 12 * c;
  float A[12];
  for (int k = 0; k < 12; ++k) A[k] = fmaf(t, A1[k], A0[k]);
  const float* mb = s->mean + 3 * (int64_t)i;
  float mu[3];
  for (int k = 0; k < 3; ++k) {
    float p = fmaf(A[4 * k + 0], mb[0], fmaf(A[4 * k + 1], mb[1], fmaf(A[4 * k + 2], mb[2], A[4 * k + 3])));
    if (d >= 1) {
      float acc = 0.0f;
      for (int r = 0; r < s->R; ++r)
        acc = fmaf(basis[r], (float)s->motion_q[((int64_t)i * s->R + r) * 3 + k], acc);
      p = fmaf(s->motion_scale[c], acc, p);
    }
    /* Eq. (1) "+ delta^(2) + delta^(3)" (reading I1): the level-l position
     * residual is applied iff the cluster's depth is >= l, added in this order in binary32 */
    if (d >= 2 && s->delta2) p = p + s->delta2[3 * (int64_t)i + k];
    if (d >= 3 && s->delta3) p = p + s->delta3[3 * (int64_t)i + k];
    mu[k] = p;
    o->mu[k] = p;
  }

  /* ---- O-3: camera transform ---- */
  const float* Rw = cam->R;
  float pc[3];
  for (int k = 0; k < 3; ++k)
    pc[k] = fmaf(Rw[3 * k + 0], mu[0], fmaf(Rw[3 * k + 1], mu[1], fmaf(Rw[3 * k + 2], mu[2], cam->t[k])));
  float z = pc[2];
  o->z = z;
  if (!(z > cam->znear)) return;
  float rz = 1.0f / z;
  float txz = pc[0] * rz;
  float tyz = pc[1] * rz;
  float limx = ((0.5f * (float)cam->W) / cam->fx) * 1.3f;
  float limy = ((0.5f * (float)cam->H) / cam->fy) * 1.3f;
  float xt = clampf(txz, -limx, limx) * z;
  float yt = clampf(tyz, -limy, limy) * z;
  /* Jacobian of the pinhole projection at the (clamped) point */
  float J00 = cam->fx * rz;
  float J02 = -(((cam->fx * xt) * rz) * rz);
  float J11 = cam->fy * rz;
  float J12 = -(((cam->fy * yt) * rz) * rz);
  /* M = J * R_wc  (2x3) */
  float M0[3], M1[3];
  for (int k = 0; k < 3; ++k) {
    M0[k] = fmaf(J02, Rw[6 + k], J00 * Rw[0 + k]);
    M1[k] = fmaf(J12, Rw[6 + k], J11 * Rw[3 + k]);
  }
  /* Sigma' = M Sigma M^T */
  const float* S6 = s->cov3d_lv ? s->cov3d_lv + 6 * ((int64_t)d * s->N + i) : s->cov3d + 6 * (int64_t)i;
  float S6t[6];
  if (s->affine_cov) {
    /* reading I4: Sigma_t = L Sigma L^T with L = the 3x3 part of A_{c,t}; binary32, this order:
     * Mm = L S (row a, column b), then Sigma_t[a][b] = Mm[a] . L[b] */
    const float Sf[9] = {S6[0], S6[1], S6[2], S6[1], S6[3], S6[4], S6[2], S6[4], S6[5]};
    float Mm[9];
    for (int a = 0; a < 3; ++a)
      for (int b = 0; b < 3; ++b)
        Mm[3 * a + b] = fmaf(A[4 * a + 2], Sf[6 + b], fmaf(A[4 * a + 1], Sf[3 + b], A[4 * a + 0] * Sf[b]));
    int o6 = 0;
    for (int a = 0; a < 3; ++a)
      for (int b = a; b < 3; ++b)
        S6t[o6++] = fmaf(Mm[3 * a + 2], A[4 * b + 2], fmaf(Mm[3 * a + 1], A[4 * b + 1], Mm[3 * a + 0] * A[4 * b + 0]));
    S6 = S6t;
  }
  float S[9] = {S6[0], S6[1], S6[2], S6[1], S6[3], S6[4], S6[2], S6[4], S6[5]};
  float v0[3], v1[3];
  for (int a = 0; a < 3; ++a) {
    v0[a] = fmaf(S[3 * a + 2], M0[2], fmaf(S[3 * a + 1], M0[1], S[3 * a + 0] * M0[0]));
    v1[a] = fmaf(S[3 * a + 2], M1[2], fmaf(S[3 * a + 1], M1[1], S[3 * a + 0] * M1[0]));
  }
  float s00 = fmaf(M0[2], v0[2], fmaf(M0[1], v0[1], M0[0] * v0[0]));
  float s01 = fmaf(M0[2], v1[2], fmaf(M0[1], v1[1], M0[0] * v1[0]));
  float s11 = fmaf(M1[2], v1[2], fmaf(M1[1], v1[1], M1[0] * v1[0]));
  float a = s00 + 0.3f, b = s01, cc = s11 + 0.3f; /* reading A11: dilation 0.3 */
  float det = fmaf(a, cc, -(b * b));
  if (!(det > 0.0f)) return;
  float rdet = 1.0f / det;
  float conic_a = cc * rdet, conic_b = -(b * rdet), conic_c = a * rdet;
  o->cov2d[0] = a; o->cov2d[1] = b; o->cov2d[2] = cc;
  o->qa = 0.5f * conic_a;
  o->qb = conic_b;
  o->qc = 0.5f * conic_c;
  float mid = 0.5f * (a + cc);
  float disc = fmaxf(0.1f, fmaf(mid, mid, -det));
  float lam = mid + sqrtf(disc);
  float rad = ceilf(3.0f * sqrtf(lam));
  o->radius = (int32_t)rad;
  float mx = fmaf(cam->fx, txz, cam->cx);
  float my = fmaf(cam->fy, tyz, cam->cy);
  o->mx = mx;
  o->my = my;
  /* tile rectangle (half-open), clamped in float before conversion (reading A15) */
  float TXf = (float)((cam->W + TILE - 1) / TILE), TYf = (float)((cam->H + TILE - 1) / TILE);
  int tx0 = (int)clampf(floorf((mx - rad) * 0.0625f), 0.0f, TXf);
  int tx1 = (int)clampf(floorf(((mx + rad) + 15.0f) * 0.0625f), 0.0f, TXf);
  int ty0 = (int)clampf(floorf((my - rad) * 0.0625f), 0.0f, TYf);
  int ty1 = (int)clampf(floorf(((my + rad) + 15.0f) * 0.0625f), 0.0f, TYf);
  if (tx1 <= tx0 || ty1 <= ty0) return;
  o->rect[0] = tx0; o->rect[1] = ty0; o->rect[2] = tx1; o->rect[3] = ty1;
  o->count = (tx1 - tx0) * (ty1 - ty0);
  memcpy(&o->depth_bits, &z, 4);

  /* ---- colour: degree-L real SH of the view direction, + level-3 residual iff d >= 3 ---- */
  double cc3[3]; /* camera centre = -R^T t */
  for (int k = 0; k < 3; ++k)
    cc3[k] = -((double)Rw[0 + k] * cam->t[0] + (double)Rw[3 + k] * cam->t[1] + (double)Rw[6 + k] * cam->t[2]);
  double dx = (double)mu[0] - cc3[0], dy = (double)mu[1] - cc3[1], dz = (double)mu[2] - cc3[2];
  double nrm = sqrt(dx * dx + dy * dy + dz * dz);
  dx /= nrm; dy /= nrm; dz /= nrm;
  double Y[16];
  sh_basis(s->K, dx, dy, dz, Y);
  for (int ch = 0; ch < 3; ++ch) {
    double acc = 0.5;
    for (int j = 0; j < s->K; ++j) {
      double coef = (double)s->sh_base[((int64_t)i * s->K + j) * 3 + ch];
      if (d >= 3) coef += (double)s->sh_res[((int64_t)i * s->K + j) * 3 + ch];
      if (s->d_sh) /* colour: base plus the learned refinements of the delivered levels */
        for (int l = 1; l <= d && l <= 3; ++l)
          coef += (double)s->d_sh[(((int64_t)(l - 1) * s->N + i) * s->K + j) * 3 + ch];
      acc += Y[j] * coef;
    }
    o->rgb[ch] = acc > 0.0 ? acc : 0.0;
  }
  o->valid = 1;
}

/* Project every Gaussian of one state.  depth: int8 [C].  out: orc_proj [N]. */
void orc_project_state(const orc_scene* s, const orc_camera* cam, float t, const int8_t* depth,
                       orc_proj* out) {
  float basis[64];
  orc_basis(t, s->R, basis);
  for (int c = 0; c < s->C; ++c)
    for (int i = s->group_off[4 * c]; i < s->group_off[4 * c + 4]; ++i)
      project_one(s, cam, t, basis, c, i, (int)depth[c], &out[i]);
}

int32_t orc_sizeof_proj(void) { return (int32_t)sizeof(orc_proj); }

/* ------------------------------------------------------------------------------------------ */
/* O-4  order: survivors sorted by (depth bits, Gaussian index)                                */
/* ------------------------------------------------------------------------------------------ */

typedef struct { uint32_t depth_bits; int32_t idx; } order_key;

static int cmp_order(const void* pa, const void* pb) {
  const order_key* a = (const order_key*)pa;
  const order_key* b = (const order_key*)pb;
  if (a->depth_bits != b->depth_bits) return a->depth_bits < b->depth_bits ? -1 : 1;
  return (a->idx > b->idx) - (a->idx < b->idx);
}

static int64_t build_order(const orc_proj* p, int32_t N, order_key* ord) {
  int64_t n = 0;
  for (int32_t i = 0; i < N; ++i)
    if (p[i].valid) {
      ord[n].depth_bits = p[i].depth_bits;
      ord[n].idx = i;
      ++n;
    }
  qsort(ord, (size_t)n, sizeof(order_key), cmp_order);
  return n;
}

/* canonical key list of one state: all (tile, depth bits, index) triples, lexicographic.
 * Returns the number of keys; writes at most cap of them. tile = ty*TX + tx. */
typedef struct { uint32_t tile, depth_bits; int32_t idx; } tile_key;

static int cmp_tile_key(const void* pa, const void* pb) {
  const tile_key* a = (const tile_key*)pa;
  const tile_key* b = (const tile_key*)pb;
  if (a->tile != b->tile) return a->tile < b->tile ? -1 : 1;
  if (a->depth_bits != b->depth_bits) return a->depth_bits < b->depth_bits ? -1 : 1;
  return (a->idx > b->idx) - (a->idx < b->idx);
}

int64_t orc_keys_state(const orc_proj* p, int32_t N, int32_t TX, int64_t cap, uint32_t* tile,
                       uint32_t* depth_bits, int32_t* idx) {
  int64_t total = 0;
  for (int32_t i = 0; i < N; ++i)
    if (p[i].valid) total += p[i].count;
  if (total > cap) return total;
  tile_key* keys = (tile_key*)malloc(sizeof(tile_key) * (size_t)(total > 0 ? total : 1));
  int64_t n = 0;
  for (int32_t i = 0; i < N; ++i)
    if (p[i].valid)
      for (int ty = p[i].rect[1]; ty < p[i].rect[3]; ++ty)
        for (int tx = p[i].rect[0]; tx < p[i].rect[2]; ++tx) {
          keys[n].tile = (uint32_t)(ty * TX + tx);
          keys[n].depth_bits = p[i].depth_bits;
          keys[n].idx = i;
          ++n;
        }
  qsort(keys, (size_t)n, sizeof(tile_key), cmp_tile_key);
  for (int64_t k = 0; k < n; ++k) {
    tile[k] = keys[k].tile;
    depth_bits[k] = keys[k].depth_bits;
    idx[k] = keys[k].idx;
  }
  free(keys);
  return n;
}

/* ------------------------------------------------------------------------------------------ */
/* O-5  pixel                                                                                  */
/* ------------------------------------------------------------------------------------------ */

/* One (pixel, Gaussian) step.  Returns 1 if the pixel terminated at this Gaussian.
 * px, py = pixel centre.  T, Cacc = the pixel's running transmittance / colour (double). */
static inline int pixel_step(const orc_proj* g, float opac, float tau, float px, float py, double t_stop,
                             double* T, double* Cacc, int64_t* evaluated, double* alpha_out) {
  /* spec-exact fp32 quadratic form: u=A dx; s=fma(B,dy,u); q=s dx; v=Cq dy; q=fma(v,dy,q) */
  float dx = g->mx - px;
  float dy = g->my - py;
  float u = g->qa * dx;
  float sacc = fmaf(g->qb, dy, u);
  float q = sacc * dx;
  float v = g->qc * dy;
  q = fmaf(v, dy, q);
  ++*evaluated;
  if (alpha_out) *alpha_out = 0.0;
  if (q > tau) return 0; /* alpha < 1/255: skipped (bit-exact decision) */
  double e = exp(-(double)q);
  double alpha = (double)opac * e;
  if (alpha > 0.99) alpha = 0.99;
  double Tn = *T * (1.0 - alpha);
  if (Tn < t_stop) return 1; /* stop; this Gaussian is NOT added */
  if (alpha_out) *alpha_out = alpha;
  double w = alpha * *T;
  Cacc[0] += w * g->rgb[0];
  Cacc[1] += w * g->rgb[1];
  Cacc[2] += w * g->rgb[2];
  *T = Tn;
  return 0;
}

/* O1: brute force.  For every pixel, walk ALL survivors in depth order; a Gaussian takes part iff
 * its tile rectangle contains the pixel's tile.  img: double [H,W,3].  stats: [0]=I_b (tile
 * intersections), [1]=E_b (pairs evaluated).  Tfinal (optional): double [H,W]. */
void orc_render_O1(const orc_scene* s, const orc_camera* cam, const orc_proj* p, double t_stop, double* img,
                   int64_t* stats, double* Tfinal) {
  order_key* ord = (order_key*)malloc(sizeof(order_key) * (size_t)(s->N > 0 ? s->N : 1));
  int64_t n = build_order(p, s->N, ord);
  int64_t inter = 0, evaluated = 0;
  for (int64_t k = 0; k < n; ++k) inter += p[ord[k].idx].count;
  for (int y = 0; y < cam->H; ++y)
    for (int x = 0; x < cam->W; ++x) {
      int tx = x / TILE, ty = y / TILE;
      float px = (float)x + 0.5f, py = (float)y + 0.5f;
      double T = 1.0, Cc[3] = {0.0, 0.0, 0.0};
      for (int64_t k = 0; k < n; ++k) {
        const orc_proj* g = &p[ord[k].idx];
        if (tx < g->rect[0] || tx >= g->rect[2] || ty < g->rect[1] || ty >= g->rect[3]) continue;
        if (pixel_step(g, g->opacity, g->tau, px, py, t_stop, &T, Cc, &evaluated, NULL))
          break;
      }
      double* o = img + 3 * ((int64_t)y * cam->W + x);
      for (int ch = 0; ch < 3; ++ch) o[ch] = Cc[ch] + T * (double)s->background[ch];
      if (Tfinal) Tfinal[(int64_t)y * cam->W + x] = T;
    }
  if (stats) { stats[0] = inter; stats[1] = evaluated; }
  free(ord);
}

/* O2: the same per-pixel arithmetic sequence, Gaussian-major: walk survivors in depth order and
 * scatter each into the pixels of its tile rectangle.  Must equal O1 bitwise (pin P11). */
void orc_render_O2(const orc_scene* s, const orc_camera* cam, const orc_proj* p, double t_stop, double* img,
                   int64_t* stats, double* Tfinal) {
  order_key* ord = (order_key*)malloc(sizeof(order_key) * (size_t)(s->N > 0 ? s->N : 1));
  int64_t n = build_order(p, s->N, ord);
  int64_t P = (int64_t)cam->W * cam->H;
  double* T = (double*)malloc(sizeof(double) * (size_t)P);
  uint8_t* done = (uint8_t*)calloc((size_t)P, 1);
  for (int64_t k = 0; k < P; ++k) T[k] = 1.0;
  memset(img, 0, sizeof(double) * 3 * (size_t)P);
  int64_t inter = 0, evaluated = 0;
  for (int64_t k = 0; k < n; ++k) {
    int gi = ord[k].idx;
    const orc_proj* g = &p[gi];
    inter += g->count;
    int x0 = g->rect[0] * TILE, x1 = g->rect[2] * TILE, y0 = g->rect[1] * TILE, y1 = g->rect[3] * TILE;
    if (x1 > cam->W) x1 = cam->W;
    if (y1 > cam->H) y1 = cam->H;
    for (int y = y0; y < y1; ++y)
      for (int x = x0; x < x1; ++x) {
        int64_t pix = (int64_t)y * cam->W + x;
        if (done[pix]) continue;
        if (pixel_step(g, g->opacity, g->tau, (float)x + 0.5f, (float)y + 0.5f, t_stop, &T[pix],
                       img + 3 * pix, &evaluated, NULL))
          done[pix] = 1;
      }
  }
  for (int64_t pix = 0; pix < P; ++pix) {
    for (int ch = 0; ch < 3; ++ch) img[3 * pix + ch] += T[pix] * (double)s->background[ch];
    if (Tfinal) Tfinal[pix] = T[pix];
  }
  if (stats) { stats[0] = inter; stats[1] = evaluated; }
  free(ord); free(T); free(done);
}

/* Per-pixel trace for pins P4/P5/P16: the sequence of Gaussians the pixel meets, with alpha
 * (0 if skipped) and T after each.  Returns the number of entries (terminating one included,
 * flagged by alpha = -1). */
int64_t orc_trace_pixel(const orc_scene* s, const orc_camera* cam, const orc_proj* p, double t_stop, int32_t x,
                        int32_t y, int64_t cap, int32_t* gidx, double* alpha, double* Tafter) {
  order_key* ord = (order_key*)malloc(sizeof(order_key) * (size_t)(s->N > 0 ? s->N : 1));
  int64_t n = build_order(p, s->N, ord);
  int tx = x / TILE, ty = y / TILE;
  double T = 1.0, Cc[3] = {0, 0, 0};
  int64_t m = 0, evaluated = 0;
  for (int64_t k = 0; k < n; ++k) {
    const orc_proj* g = &p[ord[k].idx];
    if (tx < g->rect[0] || tx >= g->rect[2] || ty < g->rect[1] || ty >= g->rect[3]) continue;
    double a = 0.0;
    int stop = pixel_step(g, g->opacity, g->tau, (float)x + 0.5f, (float)y + 0.5f,
                          t_stop, &T, Cc, &evaluated, &a);
    if (m < cap) { gidx[m] = ord[k].idx; alpha[m] = stop ? -1.0 : a; Tafter[m] = T; }
    ++m;
    if (stop) break;
  }
  free(ord);
  return m;
}

/* Batch driver (O2 per state, OpenMP over states: states are independent).  levels int8 [B,C];
 * img double [B,H,W,3]; stats int64 [B,2]. Used for parity tests and as the timed CPU baseline. */
void orc_render_batch(const orc_scene* s, const orc_camera* cam, float t, const int8_t* levels, int32_t B,
                      double t_stop, double* img, int64_t* stats, int32_t brute_force) {
  int64_t P3 = 3 * (int64_t)cam->W * cam->H;
#pragma omp parallel for schedule(dynamic, 1)
  for (int b = 0; b < B; ++b) {
    orc_proj* p = (orc_proj*)malloc(sizeof(orc_proj) * (size_t)(s->N > 0 ? s->N : 1));
    orc_project_state(s, cam, t, levels + (int64_t)b * s->C, p);
    if (brute_force)
      orc_render_O1(s, cam, p, t_stop, img + b * P3, stats ? stats + 2 * b : NULL, NULL);
    else
      orc_render_O2(s, cam, p, t_stop, img + b * P3, stats ? stats + 2 * b : NULL, NULL);
    free(p);
  }
}

int32_t orc_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

/* ------------------------------------------------------------------------------------------ */
/* O-6  distortion                                                                             */
/* ------------------------------------------------------------------------------------------ */

/* imgs: double [B, n] (n = 3*W*H), ref: double [n].  MSE in double; PSNR = -10 log10(max(MSE,1e-10)). */
void orc_distortion(const double* imgs, const double* ref, int32_t B, int64_t n, double* mse, double* psnr_db) {
  for (int b = 0; b < B; ++b) {
    double sse = 0.0;
    for (int64_t k = 0; k < n; ++k) {
      double d = imgs[(int64_t)b * n + k] - ref[k];
      sse += d * d;
    }
    mse[b] = sse / (double)n;
    double m = mse[b] > 1e-10 ? mse[b] : 1e-10;
    psnr_db[b] = -10.0 * log10(m);
  }
}

/* ------------------------------------------------------------------------------------------ */
/* O-7  counterfactual utility: Eq. (3) per pair, Eq. (4) per group          */
/* ------------------------------------------------------------------------------------------ */

static int cmp_double(const void* a, const void* b) {
  double x = *(const double*)a, y = *(const double*)b;
  return (x > y) - (x < y);
}

/* mean, Q_0.1 (linear interpolation at position 0.1 (n-1) of the sorted samples), population std,
 * and the risk-adjusted utility of Eq. (4) with alpha = 0.25, beta = 0.05. */
static void aggregate(double* v, int64_t n, double* out4) {
  if (n == 0) { out4[0] = out4[1] = out4[2] = out4[3] = 0.0; return; }
  double mean = 0.0;
  for (int64_t k = 0; k < n; ++k) mean += v[k];
  mean /= (double)n;
  double var = 0.0;
  for (int64_t k = 0; k < n; ++k) var += (v[k] - mean) * (v[k] - mean);
  var /= (double)n;
  double sd = sqrt(var);
  qsort(v, (size_t)n, sizeof(double), cmp_double);
  double pos = 0.1 * (double)(n - 1);
  int64_t lo = (int64_t)floor(pos);
  int64_t hi = lo + 1 < n ? lo + 1 : n - 1;
  double fr = pos - (double)lo;
  double q10 = v[lo] + fr * (v[hi] - v[lo]);
  const double alpha = 0.25, beta = 0.05;
  out4[0] = mean;
  out4[1] = q10;
  out4[2] = sd;
  out4[3] = ((1.0 - alpha) * mean + alpha * q10) / (1.0 + beta * sd);
}

/* mse, psnr: [B].  Pairs: idx_without[p], idx_with[p], group_id[p] in [0,G).
 * delta_mse[p] = MSE(m) - MSE(m u g) (Eq. 3 with D = MSE); delta_db[p] = PSNR(m u g) - PSNR(m).
 * util: double [G, 9] = {mean,q10,std,risk}_mse, {mean,q10,std,risk}_dB, count. */
void orc_group_utility(const double* mse, const double* psnr_db, const int32_t* idx_without,
                       const int32_t* idx_with, const int32_t* group_id, int64_t n_pairs, int32_t G,
                       double* delta_mse, double* delta_db, double* util) {
  for (int64_t p = 0; p < n_pairs; ++p) {
    delta_mse[p] = mse[idx_without[p]] - mse[idx_with[p]];
    delta_db[p] = psnr_db[idx_with[p]] - psnr_db[idx_without[p]];
  }
  double* buf = (double*)malloc(sizeof(double) * (size_t)(n_pairs > 0 ? n_pairs : 1));
  for (int g = 0; g < G; ++g) {
    int64_t n = 0;
    for (int64_t p = 0; p < n_pairs; ++p)
      if (group_id[p] == g) buf[n++] = delta_mse[p];
    aggregate(buf, n, util + 9 * g);
    n = 0;
    for (int64_t p = 0; p < n_pairs; ++p)
      if (group_id[p] == g) buf[n++] = delta_db[p];
    aggregate(buf, n, util + 9 * g + 4);
    util[9 * g + 8] = (double)n;
  }
  free(buf);
}

/* ------------------------------------------------------------------------------------------ */
/* O-8  backward of O-5: gradients of a linear functional of one state's image                  */
/* ------------------------------------------------------------------------------------------ */

/* SURVEY.md §8(f)-4's follow-on (the training objective is a function of the rendered images, so
 * its gradient enters through dL/d(image)).  Given g = dL/d(pixel) for every pixel and channel of ONE state's image
 * (e.g. 2 (I - R) / (3 W H) for L = MSE), the gradient of L with respect to the 2-D quantities of every Gaussian of
 * the state that O-5 reads: rgb[3], opacity, qa, qb, qc (= A, B, Cq), mx, my.
 *
 * Definition (the pixel of O-5 written out): with the accepted Gaussians i = 1..n of a pixel in O-4 order,
 *   alpha_i = min(0.99, o_i exp(-q_i)),  T_1 = 1,  T_{i+1} = T_i (1 - alpha_i),  pixel = sum_i alpha_i T_i c_i + T_{n+1} bg.
 * The discrete decisions — which Gaussians are evaluated (tile rectangles), the cut q > tau, the cap at 0.99 and the
 * stop T' < t_stop — are constants of the differentiation (they are piecewise constant in the parameters).  Hence
 *   dpixel/dc_i     = alpha_i T_i
 *   dpixel/dalpha_i = T_i c_i - S_i / (1 - alpha_i),   S_i = sum_{j>i} alpha_j T_j c_j + T_{n+1} bg
 *   dalpha_i/do_i   = exp(-q_i),  dalpha_i/dq_i = -alpha_i      (both 0 where the cap is active)
 *   q = (A dx + B dy) dx + Cq dy^2 with dx = mx - px, dy = my - py:
 *   dq/dA = dx^2, dq/dB = dx dy, dq/dCq = dy^2, dq/dmx = 2 A dx + B dy, dq/dmy = B dx + 2 Cq dy.
 * Brute force per pixel like O1: a forward walk that records the accepted sequence, then the sums above in double
 * from the same fp32 dx, dy, q the forward decisions use.
 *   g_img  double [H,W,3];  grad double [N,9] = (drgb[3], dopacity, dqa, dqb, dqc, dmx, dmy), zeroed here.
 *   grad_abs (optional, [N,9]): a magnitude for every entry, against which a floating-point evaluation of these
 *   strongly cancelling sums can be judged: the same sums with dL/dalpha replaced by
 *   |g| (T |c| + 2 M / (1 - alpha)), M = sum_j alpha_j T_j |c_j| + T_end |bg| (everything a pixel is made of: an
 *   implementation may form the suffix S_i as "final pixel minus prefix"), and absolute chain factors. */
void orc_backward_O1(const orc_scene* s, const orc_camera* cam, const orc_proj* p, double t_stop, const double* g_img,
                     double* grad, double* grad_abs) {
  order_key* ord = (order_key*)malloc(sizeof(order_key) * (size_t)(s->N > 0 ? s->N : 1));
  int64_t n = build_order(p, s->N, ord);
  for (int64_t k = 0; k < 9 * (int64_t)s->N; ++k) grad[k] = 0.0;
  if (grad_abs)
    for (int64_t k = 0; k < 9 * (int64_t)s->N; ++k) grad_abs[k] = 0.0;
  /* accepted sequence of one pixel */
  int32_t* a_idx = (int32_t*)malloc(sizeof(int32_t) * (size_t)(n > 0 ? n : 1));
  double* a_alpha = (double*)malloc(sizeof(double) * (size_t)(n > 0 ? n : 1));
  double* a_T = (double*)malloc(sizeof(double) * (size_t)(n > 0 ? n : 1));
  double* a_e = (double*)malloc(sizeof(double) * (size_t)(n > 0 ? n : 1));
  float* a_dx = (float*)malloc(sizeof(float) * (size_t)(n > 0 ? n : 1));
  float* a_dy = (float*)malloc(sizeof(float) * (size_t)(n > 0 ? n : 1));
  int* a_cap = (int*)malloc(sizeof(int) * (size_t)(n > 0 ? n : 1));
  for (int y = 0; y < cam->H; ++y)
    for (int x = 0; x < cam->W; ++x) {
      const int tx = x / TILE, ty = y / TILE;
      const float px = (float)x + 0.5f, py = (float)y + 0.5f;
      const double* g = g_img + 3 * ((int64_t)y * cam->W + x);
      double T = 1.0;
      int64_t m = 0;
      for (int64_t k = 0; k < n; ++k) {
        const orc_proj* gs = &p[ord[k].idx];
        if (tx < gs->rect[0] || tx >= gs->rect[2] || ty < gs->rect[1] || ty >= gs->rect[3]) continue;
        /* the forward step of O-5, decisions in fp32 */
        float dx = gs->mx - px;
        float dy = gs->my - py;
        float u = gs->qa * dx;
        float sacc = fmaf(gs->qb, dy, u);
        float q = sacc * dx;
        float v = gs->qc * dy;
        q = fmaf(v, dy, q);
        if (q > gs->tau) continue;
        double e = exp(-(double)q);
        double alpha = (double)gs->opacity * e;
        int cap = 0;
        if (alpha > 0.99) { alpha = 0.99; cap = 1; }
        double Tn = T * (1.0 - alpha);
        if (Tn < t_stop) break;
        a_idx[m] = ord[k].idx; a_alpha[m] = alpha; a_T[m] = T; a_e[m] = e; a_dx[m] = dx; a_dy[m] = dy; a_cap[m] = cap;
        ++m;
        T = Tn;
      }
      double M[3]; /* magnitude of what the pixel is made of, per channel */
      for (int ch = 0; ch < 3; ++ch) {
        M[ch] = T * fabs((double)s->background[ch]);
        for (int64_t i = 0; i < m; ++i) M[ch] += a_alpha[i] * a_T[i] * fabs(p[a_idx[i]].rgb[ch]);
      }
      /* suffix S_i, built from the back: starts as T_{n+1} bg */
      double S[3] = {T * (double)s->background[0], T * (double)s->background[1], T * (double)s->background[2]};
      for (int64_t i = m - 1; i >= 0; --i) {
        const orc_proj* gs = &p[a_idx[i]];
        double* gr = grad + 9 * (int64_t)a_idx[i];
        const double w = a_alpha[i] * a_T[i];
        double dL_dalpha = 0.0, mag = 0.0, c9[9] = {0, 0, 0, 0, 0, 0, 0, 0, 0}, m9[9] = {0, 0, 0, 0, 0, 0, 0, 0, 0};
        for (int ch = 0; ch < 3; ++ch) {
          c9[ch] = w * g[ch];
          m9[ch] = fabs(c9[ch]);
          dL_dalpha += g[ch] * (a_T[i] * gs->rgb[ch] - S[ch] / (1.0 - a_alpha[i]));
          mag += fabs(g[ch]) * (a_T[i] * fabs(gs->rgb[ch]) + 2.0 * M[ch] / (1.0 - a_alpha[i]));
        }
        if (!a_cap[i]) {
          const double dx = (double)a_dx[i], dy = (double)a_dy[i];
          const double dL_dq = -a_alpha[i] * dL_dalpha;
          c9[3] = a_e[i] * dL_dalpha;
          c9[4] = dL_dq * dx * dx;
          c9[5] = dL_dq * dx * dy;
          c9[6] = dL_dq * dy * dy;
          c9[7] = dL_dq * (2.0 * (double)gs->qa * dx + (double)gs->qb * dy);
          c9[8] = dL_dq * ((double)gs->qb * dx + 2.0 * (double)gs->qc * dy);
          const double mq = a_alpha[i] * mag;
          m9[3] = a_e[i] * mag;
          m9[4] = mq * dx * dx;
          m9[5] = mq * fabs(dx * dy);
          m9[6] = mq * dy * dy;
          m9[7] = mq * (2.0 * fabs((double)gs->qa * dx) + fabs((double)gs->qb * dy));
          m9[8] = mq * (fabs((double)gs->qb * dx) + 2.0 * fabs((double)gs->qc * dy));
        }
        for (int k = 0; k < 9; ++k) {
          gr[k] += c9[k];
          if (grad_abs) grad_abs[9 * (int64_t)a_idx[i] + k] += m9[k];
        }
        for (int ch = 0; ch < 3; ++ch) S[ch] += w * gs->rgb[ch];
      }
    }
  free(a_idx); free(a_alpha); free(a_T); free(a_e); free(a_dx); free(a_dy); free(a_cap);
  free(ord);
}


/* ------------------------------------------------------------------------------------------ */
/* O-9  backward of activation, deformation, EWA projection and SH colour       */
/* ------------------------------------------------------------------------------------------ */

/* partial derivatives of the SH basis of sh_basis() with respect to x, y, z taken as three independent variables
 * (the polynomial of each basis function differentiated term by term) */
static void sh_basis_grad(int K, double x, double y, double z, double* Yx, double* Yy, double* Yz) {
  const double pi = M_PI;
  for (int j = 0; j < K; ++j) Yx[j] = Yy[j] = Yz[j] = 0.0;
  if (K <= 1) return;
  double c1 = sqrt(3.0 / (4.0 * pi));
  Yy[1] = c1;
  Yz[2] = c1;
  Yx[3] = c1;
  if (K <= 4) return;
  double k4 = 0.5 * sqrt(15.0 / pi), k6 = 0.25 * sqrt(5.0 / pi), k8 = 0.25 * sqrt(15.0 / pi);
  Yx[4] = k4 * y;       Yy[4] = k4 * x;                            /* k4 x y           */
  Yy[5] = k4 * z;       Yz[5] = k4 * y;                            /* k4 y z           */
  Yz[6] = k6 * 6.0 * z;                                            /* k6 (3 z^2 - 1)   */
  Yx[7] = k4 * z;       Yz[7] = k4 * x;                            /* k4 x z           */
  Yx[8] = k8 * 2.0 * x; Yy[8] = -k8 * 2.0 * y;                     /* k8 (x^2 - y^2)   */
  if (K <= 9) return;
  double k9 = 0.25 * sqrt(35.0 / (2.0 * pi)), k10 = 0.5 * sqrt(105.0 / pi), k11 = 0.25 * sqrt(21.0 / (2.0 * pi));
  double k12 = 0.25 * sqrt(7.0 / pi), k14 = 0.25 * sqrt(105.0 / pi);
  Yx[9] = k9 * 6.0 * x * y;              Yy[9] = k9 * (3.0 * x * x - 3.0 * y * y);             /* k9 y (3x^2 - y^2) */
  Yx[10] = k10 * y * z;  Yy[10] = k10 * x * z;  Yz[10] = k10 * x * y;                           /* k10 x y z         */
  Yy[11] = k11 * (5.0 * z * z - 1.0);    Yz[11] = k11 * 10.0 * y * z;                           /* k11 y (5z^2 - 1)  */
  Yz[12] = k12 * (15.0 * z * z - 3.0);                                                           /* k12 (5z^3 - 3z)   */
  Yx[13] = k11 * (5.0 * z * z - 1.0);    Yz[13] = k11 * 10.0 * x * z;                           /* k11 x (5z^2 - 1)  */
  Yx[14] = k14 * 2.0 * x * z;  Yy[14] = -k14 * 2.0 * y * z;  Yz[14] = k14 * (x * x - y * y);    /* k14 (x^2 - y^2) z */
  Yx[15] = k9 * (3.0 * x * x - 3.0 * y * y);  Yy[15] = -k9 * 6.0 * x * y;                       /* k9 x (x^2 - 3y^2) */
}

/* exported for its pin (finite differences of orc_sh_basis) */
void orc_sh_basis_grad(int32_t K, double x, double y, double z, double* Yx, double* Yy, double* Yz) {
  sh_basis_grad(K, x, y, z, Yx, Yy, Yz);
}

/* One state.  For every Gaussian i present in the state (cluster depth d = depth[c] >= level(i)) and not culled by
 * z > znear / det > 0, g9[i] = dL/d(rgb[3], opacity, A, B, Cq, m_x, m_y) (O-8's layout) is carried back through
 *   colour      rgb_ch = max(0, S_ch), S_ch = 0.5 + sum_j Y_j(dir) coef_j,ch, coef = sh_base (+ sh_res iff d = 3),
 *               dir = (mu - camera centre) / |.|
 *   projection  DESIGN.md §3.3 in its written order (pc, rz, txz, the clamp, J, M = J R, Sigma' = M Sigma M^T + 0.3 I,
 *               conic = Sigma'^-1, A = conic_a / 2, B = conic_b, Cq = conic_c / 2, m = f txz + c)
 *   deformation mu = p + [d >= 1] rho, p = A_c(t) [mu_bar; 1], rho = s_c sum_r b_r q_r          (Eq. (1))
 *   activation  Sigma = M M^T, M = Rm(quat / |quat|) diag(exp(log_scale)); opacity = sigmoid(logit)  (§3.0)
 * all in double from the raw parameters.  Fixed decisions (constants of the differentiation, reading K1): presence,
 * the culls, the clamp of x/z, y/z at +-1.3 lim (a clamped coordinate passes no gradient through x~), rgb = max(0, .)
 * (no gradient where S_ch <= 0), tau, the radius and the rectangle.
 * Outputs are ACCUMULATED (+=), so that the caller sums states:
 *   g_mean [N,3], g_rho [N,3] (rho = the motion residual vector; dL/d(s_c q_{i,r,k}) = b_r g_rho[i,k]),
 *   g_ls [N,3], g_quat [N,4] (raw quaternion), g_logit [N], g_shb / g_shr [N,K,3], g_A [C,12] (A_c(t), row-major 3x4;
 *   dL/dA0 = g_A, dL/dA1 = t g_A), g_sc [C].
 * margin [N] (overwritten where the Gaussian is present): the smallest relative distance of a decision from its
 * threshold — a caller comparing against an fp32 implementation skips Gaussians whose margin is tiny.
 * The rest of the representation: position residual levels (g_delta2, g_delta3 [N,3]: dL/dmu of the
 * states that apply them), per-level colour residuals (g_dsh [3][N,K,3]: level l collects the states of depth >= l),
 * the affine on the covariance (reading I4: Su = L Sigma L^T adds (G + G^T) L Sigma to the linear part of g_A), and
 * per-level attribute refinements: ls_lv / quat_lv / logit_lv = the raw attributes per delivered depth [4][N,.] (base +
 * residuals of levels 1..d), and g_ls / g_quat / g_logit are then [4][N,.] too — the state's gradient goes to row
 * depth; the caller folds: base = sum over depths, residual level l = sum over depths >= l.
 * Returns 0, or -1 if a scene with such terms comes without the arrays they need. */
int32_t orc_project_backward_O9(const orc_scene* s, const float* log_scale, const float* quat, const float* logit,
                                const orc_camera* cam, float t, const int8_t* depth, const double* g9,
                                double* g_mean, double* g_rho, double* g_ls, double* g_quat, double* g_logit,
                                double* g_shb, double* g_shr, double* g_A, double* g_sc, double* margin,
                                const float* ls_lv, const float* quat_lv, const float* logit_lv, double* g_delta2,
                                double* g_delta3, double* g_dsh) {
  /* the full representation: a scene with per-level attribute refinements must come with its
   * raw per-depth parameters, one with position / colour residual levels with the arrays that receive their gradients */
  if ((s->cov3d_lv != 0) != (ls_lv != 0) || (ls_lv != 0) != (quat_lv != 0) || (ls_lv != 0) != (logit_lv != 0)) return -1;
  if ((s->delta2 && !g_delta2) || (s->delta3 && !g_delta3) || (s->d_sh && !g_dsh)) return -1;
  float basis_f[64];
  orc_basis(t, s->R, basis_f);
  double Rw[9], tw[3];
  for (int k = 0; k < 9; ++k) Rw[k] = (double)cam->R[k];
  for (int k = 0; k < 3; ++k) tw[k] = (double)cam->t[k];
  const double fx = cam->fx, fy = cam->fy;
  double cc3[3]; /* camera centre = -R^T t */
  for (int k = 0; k < 3; ++k) cc3[k] = -(Rw[0 + k] * tw[0] + Rw[3 + k] * tw[1] + Rw[6 + k] * tw[2]);
  const double limx = ((0.5 * (double)cam->W) / fx) * 1.3, limy = ((0.5 * (double)cam->H) / fy) * 1.3;

  for (int c = 0; c < s->C; ++c)
    for (int i = s->group_off[4 * c]; i < s->group_off[4 * c + 4]; ++i) {
      const int d = (int)depth[c];
      if (d < level_of(s, c, i)) continue;
      const double* g = g9 + 9 * (int64_t)i;
      double mg = 1e300;

      /* ================= forward, in double ================= */
      /* O-0 */
      /* raw attributes of this state's depth: the base, or base + the residuals of levels 1..d (reading I2; summed
       * in binary32 by the caller exactly as the forward oracle's activation sees them); ia = their row */
      const int64_t ia = ls_lv ? (int64_t)d * s->N + i : (int64_t)i;
      const float* ls_p = ls_lv ? ls_lv : log_scale;
      const float* qt_p = quat_lv ? quat_lv : quat;
      const float* lg_p = logit_lv ? logit_lv : logit;
      double sc3[3];
      for (int k = 0; k < 3; ++k) sc3[k] = exp((double)ls_p[3 * ia + k]);
      const double qw = qt_p[4 * ia + 0], qx = qt_p[4 * ia + 1], qy = qt_p[4 * ia + 2], qz = qt_p[4 * ia + 3];
      const double qn = sqrt(qw * qw + qx * qx + qy * qy + qz * qz);
      const double w = qw / qn, x = qx / qn, y = qy / qn, z = qz / qn;
      const double Rm[9] = {1.0 - 2.0 * (y * y + z * z), 2.0 * (x * y - w * z),       2.0 * (x * z + w * y),
                            2.0 * (x * y + w * z),       1.0 - 2.0 * (x * x + z * z), 2.0 * (y * z - w * x),
                            2.0 * (x * z - w * y),       2.0 * (y * z + w * x),       1.0 - 2.0 * (x * x + y * y)};
      double Mm[9], Sg[9]; /* Mm = Rm diag(s); Sigma = Mm Mm^T (full 3x3) */
      for (int a = 0; a < 3; ++a)
        for (int k = 0; k < 3; ++k) Mm[3 * a + k] = Rm[3 * a + k] * sc3[k];
      for (int a = 0; a < 3; ++a)
        for (int b = 0; b < 3; ++b)
          Sg[3 * a + b] = Mm[3 * a + 0] * Mm[3 * b + 0] + Mm[3 * a + 1] * Mm[3 * b + 1] + Mm[3 * a + 2] * Mm[3 * b + 2];
      const double opac = 1.0 / (1.0 + exp(-(double)lg_p[ia]));
      /* O-2 */
      double A[12];
      for (int k = 0; k < 12; ++k) A[k] = (double)s->A0[12 * c + k] + (double)t * (double)s->A1[12 * c + k];
      const double mb[3] = {s->mean[3 * (int64_t)i + 0], s->mean[3 * (int64_t)i + 1], s->mean[3 * (int64_t)i + 2]};
      double acc[3], mu[3];
      for (int k = 0; k < 3; ++k) {
        const double p = A[4 * k + 0] * mb[0] + A[4 * k + 1] * mb[1] + A[4 * k + 2] * mb[2] + A[4 * k + 3];
        acc[k] = 0.0;
        for (int r = 0; r < s->R; ++r) acc[k] += (double)basis_f[r] * (double)s->motion_q[((int64_t)i * s->R + r) * 3 + k];
        mu[k] = d >= 1 ? p + (double)s->motion_scale[c] * acc[k] : p;
        if (d >= 2 && s->delta2) mu[k] += (double)s->delta2[3 * (int64_t)i + k];
        if (d >= 3 && s->delta3) mu[k] += (double)s->delta3[3 * (int64_t)i + k];
      }
      /* reading I4 (optional): the cluster affine also transforms the covariance, Su = L Sg L^T, L = A[:, :3] */
      double Su[9], LS[9];
      for (int a = 0; a < 9; ++a) Su[a] = Sg[a];
      if (s->affine_cov) {
        for (int a = 0; a < 3; ++a)
          for (int b = 0; b < 3; ++b)
            LS[3 * a + b] = A[4 * a + 0] * Sg[0 + b] + A[4 * a + 1] * Sg[3 + b] + A[4 * a + 2] * Sg[6 + b];
        for (int a = 0; a < 3; ++a)
          for (int b = 0; b < 3; ++b)
            Su[3 * a + b] = LS[3 * a + 0] * A[4 * b + 0] + LS[3 * a + 1] * A[4 * b + 1] + LS[3 * a + 2] * A[4 * b + 2];
      }
      /* O-3 */
      double pc[3];
      for (int k = 0; k < 3; ++k) pc[k] = Rw[3 * k + 0] * mu[0] + Rw[3 * k + 1] * mu[1] + Rw[3 * k + 2] * mu[2] + tw[k];
      const double zc = pc[2];
      mg = fmin(mg, fabs(zc - (double)cam->znear) / fmax(fabs(zc), 1e-30));
      if (!(zc > (double)cam->znear)) { margin[i] = mg; continue; }
      const double rz = 1.0 / zc, txz = pc[0] * rz, tyz = pc[1] * rz;
      const int in_x = txz >= -limx && txz <= limx, in_y = tyz >= -limy && tyz <= limy;
      mg = fmin(mg, fabs(fabs(txz) - limx) / limx);
      mg = fmin(mg, fabs(fabs(tyz) - limy) / limy);
      const double cxz = in_x ? txz : (txz < 0.0 ? -limx : limx), cyz = in_y ? tyz : (tyz < 0.0 ? -limy : limy);
      const double xt = cxz * zc, yt = cyz * zc;
      const double J00 = fx * rz, J02 = -(fx * xt) * rz * rz, J11 = fy * rz, J12 = -(fy * yt) * rz * rz;
      double M0[3], M1[3], v0[3], v1[3];
      for (int k = 0; k < 3; ++k) {
        M0[k] = J00 * Rw[0 + k] + J02 * Rw[6 + k];
        M1[k] = J11 * Rw[3 + k] + J12 * Rw[6 + k];
      }
      for (int a = 0; a < 3; ++a) {
        v0[a] = Su[3 * a + 0] * M0[0] + Su[3 * a + 1] * M0[1] + Su[3 * a + 2] * M0[2];
        v1[a] = Su[3 * a + 0] * M1[0] + Su[3 * a + 1] * M1[1] + Su[3 * a + 2] * M1[2];
      }
      const double s00 = M0[0] * v0[0] + M0[1] * v0[1] + M0[2] * v0[2];
      const double s01 = M0[0] * v1[0] + M0[1] * v1[1] + M0[2] * v1[2];
      const double s11 = M1[0] * v1[0] + M1[1] * v1[1] + M1[2] * v1[2];
      const double a2 = s00 + 0.3, b2 = s01, c2 = s11 + 0.3;
      const double det = a2 * c2 - b2 * b2;
      mg = fmin(mg, fabs(det) / fmax(a2 * c2, 1e-300));
      if (!(det > 0.0)) { margin[i] = mg; continue; }
      /* colour */
      double dv[3] = {mu[0] - cc3[0], mu[1] - cc3[1], mu[2] - cc3[2]};
      const double nrm = sqrt(dv[0] * dv[0] + dv[1] * dv[1] + dv[2] * dv[2]);
      const double dir[3] = {dv[0] / nrm, dv[1] / nrm, dv[2] / nrm};
      double Y[16], Yx[16], Yy[16], Yz[16], Sch[3];
      sh_basis(s->K, dir[0], dir[1], dir[2], Y);
      sh_basis_grad(s->K, dir[0], dir[1], dir[2], Yx, Yy, Yz);
      for (int ch = 0; ch < 3; ++ch) {
        Sch[ch] = 0.5;
        for (int j = 0; j < s->K; ++j) {
          double coef = (double)s->sh_base[((int64_t)i * s->K + j) * 3 + ch];
          if (d >= 3) coef += (double)s->sh_res[((int64_t)i * s->K + j) * 3 + ch];
          if (s->d_sh)
            for (int l = 1; l <= d && l <= 3; ++l)
              coef += (double)s->d_sh[(((int64_t)(l - 1) * s->N + i) * s->K + j) * 3 + ch];
          Sch[ch] += Y[j] * coef;
        }
        mg = fmin(mg, fabs(Sch[ch]));
      }
      margin[i] = mg;

      /* ================= backward ================= */
      double dmu[3] = {0.0, 0.0, 0.0};
      /* colour: rgb_ch = max(0, S_ch) */
      {
        double dS[3], dY[16];
        for (int ch = 0; ch < 3; ++ch) dS[ch] = Sch[ch] > 0.0 ? g[ch] : 0.0;
        for (int j = 0; j < s->K; ++j) {
          dY[j] = 0.0;
          for (int ch = 0; ch < 3; ++ch) {
            double coef = (double)s->sh_base[((int64_t)i * s->K + j) * 3 + ch];
            if (d >= 3) coef += (double)s->sh_res[((int64_t)i * s->K + j) * 3 + ch];
            if (s->d_sh)
              for (int l = 1; l <= d && l <= 3; ++l) {
                coef += (double)s->d_sh[(((int64_t)(l - 1) * s->N + i) * s->K + j) * 3 + ch];
                g_dsh[(((int64_t)(l - 1) * s->N + i) * s->K + j) * 3 + ch] += Y[j] * dS[ch];
              }
            dY[j] += dS[ch] * coef;
            g_shb[((int64_t)i * s->K + j) * 3 + ch] += Y[j] * dS[ch];
            if (d >= 3) g_shr[((int64_t)i * s->K + j) * 3 + ch] += Y[j] * dS[ch];
          }
        }
        double gdir[3] = {0.0, 0.0, 0.0};
        for (int j = 0; j < s->K; ++j) {
          gdir[0] += dY[j] * Yx[j];
          gdir[1] += dY[j] * Yy[j];
          gdir[2] += dY[j] * Yz[j];
        }
        /* dir = v / |v|: d dir_a / d v_b = (delta_ab - dir_a dir_b) / |v| */
        const double dot = dir[0] * gdir[0] + dir[1] * gdir[1] + dir[2] * gdir[2];
        for (int k = 0; k < 3; ++k) dmu[k] += (gdir[k] - dir[k] * dot) / nrm;
      }
      /* opacity = sigmoid(logit) */
      g_logit[ia] += g[3] * opac * (1.0 - opac);
      /* A = conic_a / 2, B = conic_b, Cq = conic_c / 2; conic = (c, -b, a) / det, det = a c - b^2 */
      const double gca = 0.5 * g[4], gcb = g[5], gcc = 0.5 * g[6];
      const double det2 = det * det;
      const double da = gca * (-c2 * c2 / det2) + gcb * (b2 * c2 / det2) + gcc * (1.0 / det - a2 * c2 / det2);
      const double db = gca * (2.0 * b2 * c2 / det2) + gcb * (-1.0 / det - 2.0 * b2 * b2 / det2) + gcc * (2.0 * a2 * b2 / det2);
      const double dc = gca * (1.0 / det - c2 * a2 / det2) + gcb * (b2 * a2 / det2) + gcc * (-a2 * a2 / det2);
      /* a = s00 + 0.3, b = s01, c = s11 + 0.3; s00 = M0.Sigma M0, s01 = M0.Sigma M1, s11 = M1.Sigma M1 */
      double G[9], dM0[3], dM1[3]; /* G_ab = dL/dSigma_ab, the nine entries taken as independent */
      for (int a = 0; a < 3; ++a) {
        for (int b = 0; b < 3; ++b) G[3 * a + b] = da * M0[a] * M0[b] + db * M0[a] * M1[b] + dc * M1[a] * M1[b];
        dM0[a] = 2.0 * da * v0[a] + db * v1[a];
        dM1[a] = 2.0 * dc * v1[a] + db * v0[a];
      }
      if (s->affine_cov) {
        /* Su = L Sg L^T: dL/dL = (G + G^T) (L Sg) (Sg symmetric), dL/dSg = L^T G L */
        double Gs[9];
        for (int r = 0; r < 3; ++r)
          for (int cc = 0; cc < 3; ++cc) {
            double acc2 = 0.0;
            for (int q = 0; q < 3; ++q) acc2 += (G[3 * r + q] + G[3 * q + r]) * LS[3 * q + cc];
            g_A[12 * c + 4 * r + cc] += acc2;
          }
        for (int a = 0; a < 3; ++a)
          for (int b = 0; b < 3; ++b) {
            double acc2 = 0.0;
            for (int pp = 0; pp < 3; ++pp)
              for (int q = 0; q < 3; ++q) acc2 += G[3 * pp + q] * A[4 * pp + a] * A[4 * q + b];
            Gs[3 * a + b] = acc2;
          }
        for (int a = 0; a < 9; ++a) G[a] = Gs[a];
      }
      /* M0 = J00 R_0 + J02 R_2, M1 = J11 R_1 + J12 R_2 */
      double dJ00 = 0.0, dJ02 = 0.0, dJ11 = 0.0, dJ12 = 0.0;
      for (int k = 0; k < 3; ++k) {
        dJ00 += dM0[k] * Rw[0 + k];
        dJ02 += dM0[k] * Rw[6 + k];
        dJ11 += dM1[k] * Rw[3 + k];
        dJ12 += dM1[k] * Rw[6 + k];
      }
      /* J00 = fx rz, J02 = -fx xt rz^2, J11 = fy rz, J12 = -fy yt rz^2 */
      double drz = fx * dJ00 + fy * dJ11 - 2.0 * fx * xt * rz * dJ02 - 2.0 * fy * yt * rz * dJ12;
      const double dxt = -fx * rz * rz * dJ02, dyt = -fy * rz * rz * dJ12;
      /* xt = clamp(txz) zc, yt = clamp(tyz) zc; m_x = fx txz + cx, m_y = fy tyz + cy */
      double dzc = cxz * dxt + cyz * dyt;
      double dtxz = fx * g[7], dtyz = fy * g[8];
      if (in_x) dtxz += zc * dxt;
      if (in_y) dtyz += zc * dyt;
      /* txz = pc0 rz, tyz = pc1 rz, rz = 1 / zc */
      double dpc[3];
      dpc[0] = rz * dtxz;
      dpc[1] = rz * dtyz;
      drz += pc[0] * dtxz + pc[1] * dtyz;
      dzc += -rz * rz * drz;
      dpc[2] = dzc;
      /* pc = R mu + t */
      for (int k = 0; k < 3; ++k) dmu[k] += Rw[0 + k] * dpc[0] + Rw[3 + k] * dpc[1] + Rw[6 + k] * dpc[2];
      /* Eq. (1) "+ delta^(2) + delta^(3)": each applied residual moves mu one to one */
      if (d >= 2 && s->delta2) for (int k = 0; k < 3; ++k) g_delta2[3 * (int64_t)i + k] += dmu[k];
      if (d >= 3 && s->delta3) for (int k = 0; k < 3; ++k) g_delta3[3 * (int64_t)i + k] += dmu[k];
      /* Eq. (1): mu = p + [d >= 1] s_c acc, p = A [mu_bar; 1] */
      if (d >= 1) {
        for (int k = 0; k < 3; ++k) {
          g_rho[3 * (int64_t)i + k] += dmu[k];
          g_sc[c] += dmu[k] * acc[k];
        }
      }
      for (int k = 0; k < 3; ++k) {
        for (int j = 0; j < 3; ++j) {
          g_mean[3 * (int64_t)i + j] += A[4 * k + j] * dmu[k];
          g_A[12 * c + 4 * k + j] += dmu[k] * mb[j];
        }
        g_A[12 * c + 4 * k + 3] += dmu[k];
      }
      /* Sigma = Mm Mm^T, Mm = Rm diag(s), s = exp(log_scale) */
      double dMm[9], dRm[9];
      for (int a = 0; a < 3; ++a)
        for (int k = 0; k < 3; ++k) {
          dMm[3 * a + k] = 0.0;
          for (int b = 0; b < 3; ++b) dMm[3 * a + k] += (G[3 * a + b] + G[3 * b + a]) * Mm[3 * b + k];
        }
      for (int k = 0; k < 3; ++k) {
        double ds = 0.0;
        for (int a = 0; a < 3; ++a) {
          ds += dMm[3 * a + k] * Rm[3 * a + k];
          dRm[3 * a + k] = dMm[3 * a + k] * sc3[k];
        }
        g_ls[3 * ia + k] += ds * sc3[k];
      }
      /* Rm(w, x, y, z) entry by entry (the matrix written in O-0) */
      const double dw = dRm[1] * (-2.0 * z) + dRm[2] * (2.0 * y) + dRm[3] * (2.0 * z) + dRm[5] * (-2.0 * x) +
                        dRm[6] * (-2.0 * y) + dRm[7] * (2.0 * x);
      const double dx_ = dRm[1] * (2.0 * y) + dRm[2] * (2.0 * z) + dRm[3] * (2.0 * y) + dRm[4] * (-4.0 * x) +
                         dRm[5] * (-2.0 * w) + dRm[6] * (2.0 * z) + dRm[7] * (2.0 * w) + dRm[8] * (-4.0 * x);
      const double dy_ = dRm[0] * (-4.0 * y) + dRm[1] * (2.0 * x) + dRm[2] * (2.0 * w) + dRm[3] * (2.0 * x) +
                         dRm[5] * (2.0 * z) + dRm[6] * (-2.0 * w) + dRm[7] * (2.0 * z) + dRm[8] * (-4.0 * y);
      const double dz_ = dRm[0] * (-4.0 * z) + dRm[1] * (-2.0 * w) + dRm[2] * (2.0 * x) + dRm[3] * (2.0 * w) +
                         dRm[4] * (-4.0 * z) + dRm[5] * (2.0 * y) + dRm[6] * (2.0 * x) + dRm[7] * (2.0 * y);
      /* (w, x, y, z) = quat / |quat| */
      const double qd = w * dw + x * dx_ + y * dy_ + z * dz_;
      g_quat[4 * ia + 0] += (dw - w * qd) / qn;
      g_quat[4 * ia + 1] += (dx_ - x * qd) / qn;
      g_quat[4 * ia + 2] += (dy_ - y * qd) / qn;
      g_quat[4 * ia + 3] += (dz_ - z * qd) / qn;
    }
  return 0;
}
