// gsr_api.cu — the C ABI of include/gsr.h: argument checks, scene activation + upload, workspace
// carving and the launch sequence of the hot path.  No arithmetic of the method lives here except the
// load-time activation and the per-call temporal basis / camera centre, which the spec
// fixes to be evaluated once on the host in double precision and rounded to fp32.
#include <math.h>
#include <stdarg.h>
#include <stdio.h>
#include <string.h>

#include <atomic>
#include <mutex>
#include <thread>
#include <vector>

#include "gsr_internal.h"

namespace gsr {

static thread_local char g_err[512] = "";

void set_error(const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof(g_err), fmt, ap);
  va_end(ap);
}

#define GSR_CUDA(call)                                                                      \
  do {                                                                                      \
    cudaError_t e_ = (call);                                                                \
    if (e_ != cudaSuccess) {                                                                \
      set_error("%s failed: %s (%s:%d)", #call, cudaGetErrorString(e_), __FILE__, __LINE__); \
      return GSR_E_CUDA;                                                                    \
    }                                                                                       \
  } while (0)

extern thread_local int g_state_block, g_dedup;
extern std::atomic<int> g_profile;
extern std::thread::id g_profile_owner;
bool profiling_here();
void profile_reset();
// calls that enqueue a frame, currently inside the library (any thread): "profile" may only be switched while 0
static std::atomic<int> g_calls_in_flight{0};
struct InFlight {
  InFlight() { g_calls_in_flight.fetch_add(1, std::memory_order_acq_rel); }
  ~InFlight() { g_calls_in_flight.fetch_sub(1, std::memory_order_acq_rel); }
};
int profile_read(double* ms, int* n);
unsigned long long launches_total();
int measure_ffma_peak(int num_sms, double* tflops, cudaStream_t st);

// ---- optional CUDA-event timing of the memory-bound phases a1-a3 (gsr_set_option("profile", 1))
constexpr int kMaxPhaseFrames = 4096;
static cudaEvent_t g_ph[kMaxPhaseFrames][3];
static int g_ph_created = 0, g_ph_used = 0;
static int phase_slot() {
  if (!profiling_here() || g_ph_used >= kMaxPhaseFrames) return -1;
  const int slot = g_ph_used++;
  while (g_ph_created <= slot) {
    for (int k = 0; k < 3; ++k) cudaEventCreate(&g_ph[g_ph_created][k]);
    ++g_ph_created;
  }
  return slot;
}

long long default_key_capacity(int32_t N) { return 12ll * 2ll * (long long)N + (1ll << 20); }

static size_t align_up(size_t v, size_t a = 256) { return (v + a - 1) / a * a; }

// Lays the workspace out; with base == nullptr only computes the size.
size_t carve_workspace(Workspace* ws, void* base, int32_t N, int32_t C, int32_t B, int32_t tiles, long long cap) {
  char* p = (char*)base;
  size_t off = 0;
  auto take = [&](size_t bytes) -> void* {
    void* r = base ? (void*)(p + off) : nullptr;
    off += align_up(bytes);
    return r;
  };
  const size_t n_rec = 2 * (size_t)N;
  Workspace w;
  w.hdr = (WsHeader*)take(sizeof(WsHeader));
  w.depth = (int8_t*)take((size_t)(B + 1) * C);
  w.r0 = (float4*)take(sizeof(float4) * n_rec);
  w.r1 = (float4*)take(sizeof(float4) * n_rec);
  w.rc0 = (float4*)take(sizeof(float4) * n_rec);
  w.rc1 = (float4*)take(sizeof(float4) * n_rec);
  w.radius = (int32_t*)take(sizeof(int32_t) * n_rec);
  w.rect = (uint2*)take(sizeof(uint2) * n_rec);
  w.depth_bits = (uint32_t*)take(sizeof(uint32_t) * n_rec);
  w.count = (uint32_t*)take(sizeof(uint32_t) * n_rec);
  for (int k = 0; k < 2; ++k) {
    w.keys[k] = (unsigned long long*)take(sizeof(unsigned long long) * (size_t)cap);
    w.vals[k] = (uint32_t*)take(sizeof(uint32_t) * (size_t)cap);
  }
  w.tile_cursor = (uint32_t*)take(sizeof(uint32_t) * (size_t)tiles);
  w.tile_range = (uint2*)take(sizeof(uint2) * (size_t)tiles);
  w.render_range = (uint2*)take(sizeof(uint2) * (size_t)tiles);
  w.state_counts = (long long*)take(sizeof(long long) * (size_t)(B > 0 ? B : 1));
  w.sse_blk = (double*)take(sizeof(double) * (size_t)(B > 0 ? B : 1) * tiles * 8);
  w.rec = (float4*)take(sizeof(float4) * 4 * n_rec);
  w.qlist = (uint2*)take(sizeof(uint2) * 4 * (size_t)cap);
  w.qrange = (uint2*)take(sizeof(uint2) * 4 * (size_t)tiles);
  w.uorder = (uint32_t*)take(sizeof(uint32_t) * (size_t)(B > 0 ? B : 1) * tiles);
  w.upos = (uint32_t*)take(sizeof(uint32_t) * (size_t)(B > 0 ? B : 1) * tiles);
  w.n_unique = (uint32_t*)take(sizeof(uint32_t) * (size_t)tiles);
  w.work_counter = (uint32_t*)take(sizeof(uint32_t));
  w.bytes = off;
  if (ws) *ws = w;
  return off;
}

struct SceneImpl {
  DeviceScene d;
  void* blob = nullptr;  // one device allocation holding every array
};

static bool camera_ok(const gsr_camera* cam) {
  return cam && cam->W > 0 && cam->H > 0 && cam->W <= 65535 * kTile && cam->H <= 65535 * kTile && cam->fx > 0 &&
         cam->fy > 0 && 3ull * (unsigned long long)cam->W * (unsigned long long)cam->H < (1ull << 32);  // floats per image fit 32 bits
}

static void make_frame(const SceneImpl* s, const gsr_camera* cam, float t, FrameParams* fp) {
  memcpy(fp->R, cam->R_wc, sizeof(fp->R));
  memcpy(fp->t, cam->t_wc, sizeof(fp->t));
  fp->fx = cam->fx; fp->fy = cam->fy; fp->cx = cam->cx; fp->cy = cam->cy;
  fp->W = cam->W; fp->H = cam->H;
  fp->TX = (cam->W + kTile - 1) / kTile;
  fp->TY = (cam->H + kTile - 1) / kTile;
  fp->znear = cam->znear;
  fp->time = t;
  // temporal basis b_r(t) = cos(pi r t), r = 1..R (reading A6): double -> fp32 once per call
  for (int r = 0; r < GSR_MAX_R; ++r)
    fp->basis[r] = r < s->d.R ? (float)cos(M_PI * (double)(r + 1) * (double)t) : 0.0f;
  // camera centre -R^T t in double -> fp32 (colour only)
  for (int k = 0; k < 3; ++k) {
    double c = -((double)cam->R_wc[0 + k] * cam->t_wc[0] + (double)cam->R_wc[3 + k] * cam->t_wc[1] +
                 (double)cam->R_wc[6 + k] * cam->t_wc[2]);
    fp->cam_centre[k] = (float)c;
  }
  for (int k = 0; k < 3; ++k) fp->bg[k] = s->d.bg[k];
}

// DESIGN.md §3.0 activation of one Gaussian, double precision, this operation order
static void activate_one(const float ls[3], const float q[4], float logit, float cov[6], float* opac, float* tau) {
  double s[3];
  for (int k = 0; k < 3; ++k) s[k] = exp((double)ls[k]);
  double qw_ = q[0], qx = q[1], qy = q[2], qz = q[3];
  const double nrm = sqrt(qw_ * qw_ + qx * qx + qy * qy + qz * qz);
  qw_ /= nrm; qx /= nrm; qy /= nrm; qz /= nrm;
  const double Rm[9] = {1.0 - 2.0 * (qy * qy + qz * qz), 2.0 * (qx * qy - qw_ * qz), 2.0 * (qx * qz + qw_ * qy),
                        2.0 * (qx * qy + qw_ * qz), 1.0 - 2.0 * (qx * qx + qz * qz), 2.0 * (qy * qz - qw_ * qx),
                        2.0 * (qx * qz - qw_ * qy), 2.0 * (qy * qz + qw_ * qx), 1.0 - 2.0 * (qx * qx + qy * qy)};
  double M[9];
  for (int a = 0; a < 3; ++a)
    for (int k = 0; k < 3; ++k) M[3 * a + k] = Rm[3 * a + k] * s[k];
  int o = 0;
  for (int a = 0; a < 3; ++a)
    for (int b = a; b < 3; ++b) {
      double acc = M[3 * a + 0] * M[3 * b + 0];
      acc += M[3 * a + 1] * M[3 * b + 1];
      acc += M[3 * a + 2] * M[3 * b + 2];
      cov[o++] = (float)acc;
    }
  *opac = (float)(1.0 / (1.0 + exp(-(double)logit)));
  *tau = (float)log(255.0 * (double)*opac);
}

}  // namespace gsr

namespace gsr {
// The per-device error word of the index checks (gsr_internal.h): allocated on first use, zeroed once.
int* device_error_word() {
  constexpr int kMaxDev = 64;
  static std::mutex mu;
  static int* words[kMaxDev] = {};
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDev) return nullptr;
  std::lock_guard<std::mutex> lock(mu);
  if (!words[dev]) {
    int* p = nullptr;
    if (cudaMalloc(&p, sizeof(int)) != cudaSuccess) return nullptr;
    if (cudaMemset(p, 0, sizeof(int)) != cudaSuccess) { cudaFree(p); return nullptr; }
    words[dev] = p;
  }
  return words[dev];
}

}  // namespace gsr

using namespace gsr;

extern "C" {

struct gsr_scene {
  SceneImpl impl;
};

const char* gsr_last_error(void) { return g_err; }
const char* gsr_version(void) { return "gsr 0.1 sm_100a"; }

int gsr_set_option(const char* name, int value) {
  if (name && strcmp(name, "state_block") == 0 && (value == 0 || value == 1 || (value >= 4 && value <= 8) || value == 16)) {
    g_state_block = value;
    return GSR_OK;
  }
  if (name && strcmp(name, "dedup") == 0) {
    g_dedup = value != 0;
    return GSR_OK;
  }
  if (name && strcmp(name, "profile") == 0) {
    if (g_calls_in_flight.load(std::memory_order_acquire) != 0) {
      set_error("gsr_set_option: \"profile\" cannot be switched while another thread is inside a render call");
      return GSR_E_INVALID_ARG;
    }
    g_profile.store(0, std::memory_order_release);
    profile_reset();
    g_ph_used = 0;
    if (value != 0) {
      g_profile_owner = std::this_thread::get_id();
      g_profile.store(1, std::memory_order_release);
    }
    return GSR_OK;
  }
  set_error("gsr_set_option: unknown option or value");
  return GSR_E_INVALID_ARG;
}

int gsr_profile_read(double* composite_ms, int32_t* composite_launches) {
  if (!composite_ms || !composite_launches) { set_error("gsr_profile_read: NULL argument"); return GSR_E_INVALID_ARG; }
  int n = 0;
  if (profile_read(composite_ms, &n) != 0) { set_error("gsr_profile_read: event query failed"); return GSR_E_CUDA; }
  *composite_launches = n;
  profile_reset();
  return GSR_OK;
}

int gsr_profile_read_phases(double* project_ms, double* sort_ms, int32_t* frames) {
  if (!project_ms || !sort_ms || !frames) { set_error("gsr_profile_read_phases: NULL argument"); return GSR_E_INVALID_ARG; }
  double p = 0, q = 0;
  for (int k = 0; k < g_ph_used; ++k) {
    float a = 0, b = 0;
    GSR_CUDA(cudaEventSynchronize(g_ph[k][2]));
    GSR_CUDA(cudaEventElapsedTime(&a, g_ph[k][0], g_ph[k][1]));
    GSR_CUDA(cudaEventElapsedTime(&b, g_ph[k][1], g_ph[k][2]));
    p += a; q += b;
  }
  *project_ms = p; *sort_ms = q; *frames = g_ph_used;
  g_ph_used = 0;
  return GSR_OK;
}

int64_t gsr_launch_count(void) { return (int64_t)launches_total(); }

int gsr_measure_fp32_peak(double* tflops, void* cuda_stream) {
  if (!tflops) { set_error("gsr_measure_fp32_peak: NULL argument"); return GSR_E_INVALID_ARG; }
  int dev = 0, sms = 0;
  GSR_CUDA(cudaGetDevice(&dev));
  GSR_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  if (measure_ffma_peak(sms, tflops, (cudaStream_t)cuda_stream) != 0) {
    set_error("gsr_measure_fp32_peak: kernel failed: %s", cudaGetErrorString(cudaGetLastError()));
    return GSR_E_CUDA;
  }
  return GSR_OK;
}

int gsr_load_scene(const gsr_scene_desc* d, gsr_scene** out) {
  if (out) *out = nullptr;
  if (!d || !out) { set_error("gsr_load_scene: NULL argument"); return GSR_E_INVALID_ARG; }
  if (d->C <= 0 || d->C > kMaxC || d->N < 0 || d->sh_degree < 0 || d->sh_degree > GSR_MAX_SH_DEGREE || d->R < 1 ||
      d->R > GSR_MAX_R || d->N > (1 << 28)) {
    set_error("gsr_load_scene: unsupported sizes C=%d N=%d sh_degree=%d R=%d", d->C, d->N, d->sh_degree, d->R);
    return GSR_E_INVALID_ARG;
  }
  if (!d->group_off || !d->A0 || !d->A1 || !d->motion_scale ||
      (d->N > 0 && (!d->mean || !d->log_scale || !d->quat || !d->opacity_logit || !d->sh_base || !d->sh_res ||
                    !d->motion_q))) {
    set_error("gsr_load_scene: NULL array");
    return GSR_E_INVALID_ARG;
  }
  const int C = d->C, N = d->N, K = (d->sh_degree + 1) * (d->sh_degree + 1), R = d->R;
  if (d->group_off[0] != 0 || d->group_off[4 * C] != N) {
    set_error("gsr_load_scene: group_off must start at 0 and end at N");
    return GSR_E_INVALID_ARG;
  }
  for (int g = 0; g < 4 * C; ++g)
    if (d->group_off[g + 1] < d->group_off[g]) {
      set_error("gsr_load_scene: group_off not monotone at %d", g);
      return GSR_E_INVALID_ARG;
    }
  const int n_sh4 = (3 * K + 3) / 4, n_qw = (3 * R + 3) / 4;
  const size_t Np = (size_t)(N > 0 ? N : 1);

  // ---- host staging in the device layout
  std::vector<float4> g0(Np), g1(Np), g2(Np), shb((size_t)n_sh4 * Np), shr((size_t)n_sh4 * Np);
  std::vector<uint32_t> qw((size_t)n_qw * Np, 0u);
  std::vector<float4> rawq(Np), rawl(Np);
  for (int c = 0; c < C; ++c)
    for (int l = 0; l < 4; ++l)
      for (int i = d->group_off[4 * c + l]; i < d->group_off[4 * c + l + 1]; ++i) {
        float cov[6], opac, tau;
        activate_one(d->log_scale + 3 * (size_t)i, d->quat + 4 * (size_t)i, d->opacity_logit[i], cov, &opac, &tau);
        const uint32_t bits = ((uint32_t)c << 2) | (uint32_t)l;
        float bitsf;
        memcpy(&bitsf, &bits, 4);
        g0[i] = make_float4(d->mean[3 * (size_t)i], d->mean[3 * (size_t)i + 1], d->mean[3 * (size_t)i + 2], opac);
        g1[i] = make_float4(cov[0], cov[1], cov[2], tau);
        g2[i] = make_float4(cov[3], cov[4], cov[5], bitsf);
        rawq[i] = make_float4(d->quat[4 * (size_t)i], d->quat[4 * (size_t)i + 1], d->quat[4 * (size_t)i + 2], d->quat[4 * (size_t)i + 3]);
        rawl[i] = make_float4(d->log_scale[3 * (size_t)i], d->log_scale[3 * (size_t)i + 1], d->log_scale[3 * (size_t)i + 2], d->opacity_logit[i]);
        for (int w4 = 0; w4 < n_sh4; ++w4) {
          float vb[4] = {0, 0, 0, 0}, vr[4] = {0, 0, 0, 0};
          for (int e = 0; e < 4; ++e) {
            const int flat = 4 * w4 + e;
            if (flat < 3 * K) {
              vb[e] = d->sh_base[(size_t)i * 3 * K + flat];
              vr[e] = d->sh_res[(size_t)i * 3 * K + flat];
            }
          }
          shb[(size_t)w4 * Np + i] = make_float4(vb[0], vb[1], vb[2], vb[3]);
          shr[(size_t)w4 * Np + i] = make_float4(vr[0], vr[1], vr[2], vr[3]);
        }
        for (int byte = 0; byte < 3 * R; ++byte) {
          const uint32_t v = (uint8_t)d->motion_q[(size_t)i * 3 * R + byte];
          qw[(size_t)(byte >> 2) * Np + i] |= v << ((byte & 3) * 8);
        }
      }

  // ---- one device blob
  gsr_scene* sc = new (std::nothrow) gsr_scene();
  if (!sc) { set_error("gsr_load_scene: out of host memory"); return GSR_E_INVALID_ARG; }
  DeviceScene& D = sc->impl.d;
  D.C = C; D.N = N; D.K = K; D.R = R; D.sh_degree = d->sh_degree; D.n_sh4 = n_sh4; D.n_qw = n_qw;
  const bool has_attr = d->d_log_scale || d->d_quat || d->d_opacity_logit;
  const bool has_dsh = d->d_sh != nullptr;
  const bool has_delta = d->delta2 || d->delta3 || has_attr || has_dsh;  // 4 records per Gaussian
  D.V = has_delta ? 4 : 2;
  D.affine_cov = d->affine_on_covariance != 0;
  D.delta = nullptr; D.g1v = nullptr; D.g2v = nullptr; D.opv = nullptr; D.d_sh = nullptr;
  D.raw_quat_v = nullptr; D.raw_ls_v = nullptr;
  D.has_delta2 = d->delta2 != nullptr; D.has_delta3 = d->delta3 != nullptr;
  for (int k = 0; k < 3; ++k) D.bg[k] = d->background[k];
  size_t off = 0;
  auto reserve = [&](size_t bytes) { size_t o = off; off += align_up(bytes); return o; };
  const size_t o_g0 = reserve(sizeof(float4) * Np), o_g1 = reserve(sizeof(float4) * Np),
               o_g2 = reserve(sizeof(float4) * Np), o_shb = reserve(sizeof(float4) * n_sh4 * Np),
               o_shr = reserve(sizeof(float4) * n_sh4 * Np), o_qw = reserve(sizeof(uint32_t) * n_qw * Np),
               o_A0 = reserve(sizeof(float) * 12 * C), o_A1 = reserve(sizeof(float) * 12 * C),
               o_ms = reserve(sizeof(float) * C), o_go = reserve(sizeof(int32_t) * (4 * C + 1)),
               o_rq = reserve(sizeof(float4) * Np), o_rl = reserve(sizeof(float4) * Np),
               o_dl = reserve(has_delta ? sizeof(float) * 6 * Np : 0),
               o_g1v = reserve(has_attr ? sizeof(float4) * 4 * Np : 0), o_g2v = reserve(has_attr ? sizeof(float4) * 4 * Np : 0),
               o_opv = reserve(has_attr ? sizeof(float) * 4 * Np : 0),
               o_rqv = reserve(has_attr ? sizeof(float4) * 4 * Np : 0), o_rlv = reserve(has_attr ? sizeof(float4) * 4 * Np : 0),
               o_dsh = reserve(has_dsh ? sizeof(float4) * 3 * n_sh4 * Np : 0);
  cudaError_t e = cudaMalloc(&sc->impl.blob, off);
  if (e != cudaSuccess) {
    set_error("gsr_load_scene: cudaMalloc(%zu) failed: %s", off, cudaGetErrorString(e));
    delete sc;
    return GSR_E_CUDA;
  }
  char* base = (char*)sc->impl.blob;
  D.g0 = (float4*)(base + o_g0); D.g1 = (float4*)(base + o_g1); D.g2 = (float4*)(base + o_g2);
  D.sh_base = (float4*)(base + o_shb); D.sh_res = (float4*)(base + o_shr); D.qw = (uint32_t*)(base + o_qw);
  D.A0 = (float*)(base + o_A0); D.A1 = (float*)(base + o_A1); D.mscale = (float*)(base + o_ms);
  D.group_off = (int32_t*)(base + o_go);
  D.raw_quat = (float4*)(base + o_rq); D.raw_ls = (float4*)(base + o_rl);
  if (has_delta) D.delta = (float*)(base + o_dl);
  if (has_dsh) D.d_sh = (float4*)(base + o_dsh);
  if (has_attr) {
    D.g1v = (float4*)(base + o_g1v); D.g2v = (float4*)(base + o_g2v); D.opv = (float*)(base + o_opv);
    D.raw_quat_v = (float4*)(base + o_rqv); D.raw_ls_v = (float4*)(base + o_rlv);
  }
  bool ok = true;
  auto up = [&](void* dst, const void* src, size_t bytes) {
    if (bytes && cudaMemcpy(dst, src, bytes, cudaMemcpyHostToDevice) != cudaSuccess) ok = false;
  };
  up(D.g0, g0.data(), sizeof(float4) * Np); up(D.g1, g1.data(), sizeof(float4) * Np);
  up(D.g2, g2.data(), sizeof(float4) * Np);
  up(D.sh_base, shb.data(), sizeof(float4) * n_sh4 * Np); up(D.sh_res, shr.data(), sizeof(float4) * n_sh4 * Np);
  up(D.qw, qw.data(), sizeof(uint32_t) * n_qw * Np);
  up(D.raw_quat, rawq.data(), sizeof(float4) * Np); up(D.raw_ls, rawl.data(), sizeof(float4) * Np);
  up(D.A0, d->A0, sizeof(float) * 12 * C); up(D.A1, d->A1, sizeof(float) * 12 * C);
  up(D.mscale, d->motion_scale, sizeof(float) * C); up(D.group_off, d->group_off, sizeof(int32_t) * (4 * C + 1));
  if (has_delta) {  // SoA [6][N]: delta2.xyz, delta3.xyz; a missing array is zero (reading I1)
    std::vector<float> dl(6 * Np, 0.0f);
    for (int i = 0; i < N; ++i)
      for (int k = 0; k < 3; ++k) {
        if (d->delta2) dl[(size_t)k * Np + i] = d->delta2[3 * (size_t)i + k];
        if (d->delta3) dl[(size_t)(3 + k) * Np + i] = d->delta3[3 * (size_t)i + k];
      }
    up(D.delta, dl.data(), sizeof(float) * 6 * Np);
  }
  if (has_dsh) {  // [3][n_sh4][N] float4 words of the flat coefficient index j*3+ch, zero padded (as sh_base)
    std::vector<float4> ds((size_t)3 * n_sh4 * Np, make_float4(0.f, 0.f, 0.f, 0.f));
    for (int l = 0; l < 3; ++l)
      for (int i = 0; i < N; ++i)
        for (int w4 = 0; w4 < n_sh4; ++w4) {
          float v[4] = {0, 0, 0, 0};
          for (int e = 0; e < 4; ++e) {
            const int flat = 4 * w4 + e;
            if (flat < 3 * K) v[e] = d->d_sh[((size_t)l * N + i) * 3 * K + flat];
          }
          ds[((size_t)l * n_sh4 + w4) * Np + i] = make_float4(v[0], v[1], v[2], v[3]);
        }
    up(D.d_sh, ds.data(), sizeof(float4) * 3 * n_sh4 * Np);
  }
  if (has_attr) {  // per-depth attributes: base + levels 1..v in binary32 (level order), then §3.0 (reading I2)
    std::vector<float4> a1(4 * Np), a2(4 * Np), rqv(4 * Np), rlv(4 * Np);
    std::vector<float> ao(4 * Np);
    for (int i = 0; i < N; ++i) {
      float ls[3] = {d->log_scale[3 * (size_t)i], d->log_scale[3 * (size_t)i + 1], d->log_scale[3 * (size_t)i + 2]};
      float q[4] = {d->quat[4 * (size_t)i], d->quat[4 * (size_t)i + 1], d->quat[4 * (size_t)i + 2], d->quat[4 * (size_t)i + 3]};
      float lg = d->opacity_logit[i];
      for (int v = 0; v < 4; ++v) {
        if (v >= 1) {
          const size_t l = (size_t)(v - 1);
          if (d->d_log_scale) for (int k = 0; k < 3; ++k) ls[k] = ls[k] + d->d_log_scale[(l * N + i) * 3 + k];
          if (d->d_quat) for (int k = 0; k < 4; ++k) q[k] = q[k] + d->d_quat[(l * N + i) * 4 + k];
          if (d->d_opacity_logit) lg = lg + d->d_opacity_logit[l * N + i];
        }
        float cov[6], opac, tau;
        activate_one(ls, q, lg, cov, &opac, &tau);
        rqv[(size_t)v * Np + i] = make_float4(q[0], q[1], q[2], q[3]);   // raw, for the backward of the activation
        rlv[(size_t)v * Np + i] = make_float4(ls[0], ls[1], ls[2], lg);
        a1[(size_t)v * Np + i] = make_float4(cov[0], cov[1], cov[2], tau);
        a2[(size_t)v * Np + i] = make_float4(cov[3], cov[4], cov[5], 0.0f);
        ao[(size_t)v * Np + i] = opac;
      }
    }
    up(D.g1v, a1.data(), sizeof(float4) * 4 * Np); up(D.g2v, a2.data(), sizeof(float4) * 4 * Np);
    up(D.raw_quat_v, rqv.data(), sizeof(float4) * 4 * Np); up(D.raw_ls_v, rlv.data(), sizeof(float4) * 4 * Np);
    up(D.opv, ao.data(), sizeof(float) * 4 * Np);
  }
  if (!ok) {
    set_error("gsr_load_scene: upload failed: %s", cudaGetErrorString(cudaGetLastError()));
    cudaFree(sc->impl.blob);
    delete sc;
    return GSR_E_CUDA;
  }
  *out = sc;
  return GSR_OK;
}

void gsr_free_scene(gsr_scene* scene) {
  if (!scene) return;
  if (scene->impl.blob) cudaFree(scene->impl.blob);
  delete scene;
}

size_t gsr_workspace_bytes_ex(const gsr_scene* scene, const gsr_camera* cam, int32_t B, int64_t key_capacity) {
  if (!scene || !camera_ok(cam) || B < 0) return 0;
  const int tiles = ((cam->W + kTile - 1) / kTile) * ((cam->H + kTile - 1) / kTile);
  const long long cap = key_capacity > 0 ? key_capacity : default_key_capacity(rec_half(scene->impl.d));
  if (cap >= (1ll << 31)) return 0;
  return carve_workspace(nullptr, nullptr, rec_half(scene->impl.d), scene->impl.d.C, B, tiles, cap);
}

size_t gsr_workspace_bytes(const gsr_scene* scene, const gsr_camera* cam, int32_t B) {
  return gsr_workspace_bytes_ex(scene, cam, B, 0);
}

// Recovers the key capacity a workspace of ws_bytes can hold (largest cap whose layout fits).
static long long capacity_for(const gsr_scene* scene, int tiles, int32_t B, size_t ws_bytes) {
  const int N = rec_half(scene->impl.d), C = scene->impl.d.C;
  const long long dflt = default_key_capacity(N);
  if (carve_workspace(nullptr, nullptr, N, C, B, tiles, dflt) <= ws_bytes) {
    // grow while it fits (callers that passed gsr_workspace_bytes_ex with a larger capacity)
    long long lo = dflt, hi = (1ll << 31) - 1;
    while (lo < hi) {
      long long mid = lo + (hi - lo + 1) / 2;
      if (carve_workspace(nullptr, nullptr, N, C, B, tiles, mid) <= ws_bytes) lo = mid; else hi = mid - 1;
    }
    return lo;
  }
  long long lo = 0, hi = dflt;
  while (lo < hi) {
    long long mid = lo + (hi - lo + 1) / 2;
    if (carve_workspace(nullptr, nullptr, N, C, B, tiles, mid) <= ws_bytes) lo = mid; else hi = mid - 1;
  }
  return lo;
}

// a0..a3 for one frame: validates levels, projects every variant once, bins and sorts.  On success
// *ws_out / *fp_out describe the prepared frame.
static int prepare_frame(const gsr_scene* scene, const gsr_camera* cam, float t, const int8_t* levels, int32_t B,
                         void* workspace, size_t ws_bytes, cudaStream_t st, Workspace* ws_out, FrameParams* fp_out) {
  if (!scene || !camera_ok(cam) || B < 0 || (B > 0 && !levels) || !workspace) {
    set_error("gsr_render_states: invalid argument");
    return GSR_E_INVALID_ARG;
  }
  if (((uintptr_t)workspace & 255u) != 0) { set_error("gsr_render_states: workspace must be 256-byte aligned"); return GSR_E_INVALID_ARG; }
  const SceneImpl* s = &scene->impl;
  make_frame(s, cam, t, fp_out);
  const int tiles = fp_out->TX * fp_out->TY;
  if (carve_workspace(nullptr, nullptr, rec_half(s->d), s->d.C, B, tiles, 1) > ws_bytes) {
    set_error("gsr_render_states: workspace of %zu bytes is too small", ws_bytes);
    return GSR_E_WORKSPACE_TOO_SMALL;
  }
  const long long cap = capacity_for(scene, tiles, B, ws_bytes);
  if (cap < 1) { set_error("gsr_render_states: workspace too small"); return GSR_E_WORKSPACE_TOO_SMALL; }
  carve_workspace(ws_out, workspace, rec_half(s->d), s->d.C, B, tiles, cap);
  launch_init_header(*ws_out, B, s->d.C, s->d.N, *fp_out, cap, st);
  launch_validate_levels(levels, B, s->d.C, *ws_out, st);   // a0
  const int ph = phase_slot();
  if (ph >= 0) cudaEventRecord(g_ph[ph][0], st);
  launch_project(s->d, *fp_out, *ws_out, st);                // a1 + a2
  if (ph >= 0) cudaEventRecord(g_ph[ph][1], st);
  launch_bin_and_sort(s->d, *fp_out, *ws_out, cap, st);      // a3
  if (ph >= 0) cudaEventRecord(g_ph[ph][2], st);
  return GSR_OK;
}

int gsr_render_states_ex(const gsr_scene* scene, const gsr_camera* cam, float t, const int8_t* levels, int32_t B,
                         float* out, const float* ref, double* mse, float* psnr_db, void* workspace,
                         size_t ws_bytes, void* cuda_stream) {
  if (ref && !mse) { set_error("gsr_render_states: ref given without mse"); return GSR_E_INVALID_ARG; }
  cudaStream_t st = (cudaStream_t)cuda_stream;
  InFlight guard;
  Workspace ws;
  FrameParams fp;
  int rc = prepare_frame(scene, cam, t, levels, B, workspace, ws_bytes, st, &ws, &fp);
  if (rc != GSR_OK) return rc;
  launch_composite(scene->impl.d, fp, ws, ws.depth, B, out, ref, mse, psnr_db, st);  // a4 (+ fused a5)
  GSR_CUDA(cudaGetLastError());
  return GSR_OK;
}

int gsr_render_states_vs_full(const gsr_scene* scene, const gsr_camera* cam, float t, const int8_t* levels,
                              int32_t B, float* out, float* ref_out, double* mse, float* psnr_db, void* workspace,
                              size_t ws_bytes, void* cuda_stream) {
  if (!ref_out || !mse) { set_error("gsr_render_states_vs_full: ref_out and mse are required"); return GSR_E_INVALID_ARG; }
  cudaStream_t st = (cudaStream_t)cuda_stream;
  InFlight guard;
  Workspace ws;
  FrameParams fp;
  int rc = prepare_frame(scene, cam, t, levels, B, workspace, ws_bytes, st, &ws, &fp);
  if (rc != GSR_OK) return rc;
  const DeviceScene& d = scene->impl.d;
  // the reference: the full state (row B of ws.depth), composited from the same sorted lists
  launch_composite(d, fp, ws, ws.depth + (size_t)B * d.C, 1, ref_out, nullptr, nullptr, nullptr, st);
  launch_composite(d, fp, ws, ws.depth, B, out, ref_out, mse, psnr_db, st);
  GSR_CUDA(cudaGetLastError());
  return GSR_OK;
}

int gsr_render_states(const gsr_scene* scene, const gsr_camera* cam, float t, const int8_t* levels, int32_t B,
                      float* out, void* workspace, size_t ws_bytes, void* cuda_stream) {
  if (!out) { set_error("gsr_render_states: out is NULL (use gsr_render_states_ex for distortion only)"); return GSR_E_INVALID_ARG; }
  return gsr_render_states_ex(scene, cam, t, levels, B, out, nullptr, nullptr, nullptr, workspace, ws_bytes,
                              cuda_stream);
}

int64_t gsr_num_records(const gsr_scene* scene) {
  return scene ? (int64_t)scene->impl.d.N * scene->impl.d.V : 0;
}

int gsr_render_backward(const gsr_scene* scene, void* workspace, const float* images, const float* dL_dimages,
                        int32_t B, float* grad, void* cuda_stream) {
  cudaStream_t st = (cudaStream_t)cuda_stream;
  if (!scene || !workspace || B < 0 || (B > 0 && (!images || !dL_dimages)) || !grad) {
    set_error("gsr_render_backward: invalid argument");
    return GSR_E_INVALID_ARG;
  }
  if (((uintptr_t)grad & 15u) != 0) {  // rows of 12 floats are added with 16-byte vector reductions
    set_error("gsr_render_backward: grad must be 16-byte aligned");
    return GSR_E_INVALID_ARG;
  }
  // the header is read on the host: the forward call that filled the workspace has to be complete on this stream
  WsHeader h;
  GSR_CUDA(cudaMemcpyAsync(&h, workspace, sizeof(h), cudaMemcpyDeviceToHost, st));
  GSR_CUDA(cudaStreamSynchronize(st));
  if (h.N != scene->impl.d.N || h.C != scene->impl.d.C || h.B != B) {
    set_error("gsr_render_backward: the workspace does not hold a forward render of this scene with B = %d states", B);
    return GSR_E_INVALID_ARG;
  }
  if (h.status != GSR_OK) { set_error("gsr_render_backward: the forward render failed (status %d)", h.status); return h.status; }
  Workspace ws;
  carve_workspace(&ws, workspace, rec_half(scene->impl.d), h.C, h.B, h.TX * h.TY, h.key_capacity);
  launch_backward(scene->impl.d, h, ws, images, dL_dimages, grad, st);
  GSR_CUDA(cudaGetLastError());
  return GSR_OK;
}

int gsr_objective_weights(const double* d, int32_t n, double w_mean, double w_cvar, double alpha,
                          const int32_t* idx_prev, const int32_t* idx_next, int32_t n_pairs, double w_mono,
                          double* weights, void* cuda_stream) {
  if (n < 0 || n_pairs < 0 || (n > 0 && (!d || !weights)) || (n_pairs > 0 && (!idx_prev || !idx_next)) ||
      !(alpha > 0.0 && alpha <= 1.0)) {
    set_error("gsr_objective_weights: invalid argument");
    return GSR_E_INVALID_ARG;
  }
  launch_objective_weights(d, n, w_mean, w_cvar, alpha, idx_prev, idx_next, n_pairs, w_mono, weights,
                           (cudaStream_t)cuda_stream);
  GSR_CUDA(cudaGetLastError());
  return GSR_OK;
}

int gsr_flicker_backward(const float* imgs_t1, const float* imgs_t2, const float* ref_t1, const float* ref_t2, int32_t B,
                         int32_t H, int32_t W, const double* weight, float* g_t1, float* g_t2, void* cuda_stream) {
  if (B < 0 || H <= 0 || W <= 0 || (B > 0 && (!imgs_t1 || !imgs_t2 || !ref_t1 || !ref_t2 || (!g_t1 && !g_t2)))) {
    set_error("gsr_flicker_backward: invalid argument");
    return GSR_E_INVALID_ARG;
  }
  launch_flicker_backward(imgs_t1, imgs_t2, ref_t1, ref_t2, B, H, W, weight, g_t1, g_t2, (cudaStream_t)cuda_stream);
  GSR_CUDA(cudaGetLastError());
  return GSR_OK;
}

size_t gsr_distortion_backward_workspace_bytes(int32_t H, int32_t W) {
  if (H <= 0 || W <= 0) return 0;
  return align_up(sizeof(double) * 2 * 3 * (size_t)H * (size_t)W);
}

int gsr_distortion_backward(const float* imgs, const float* ref, int32_t B, int32_t H, int32_t W, const double* weight,
                            double lambda_ssim, float* dL_dimgs, void* workspace, size_t ws_bytes, void* cuda_stream) {
  if (B < 0 || H <= 0 || W <= 0 || (B > 0 && (!imgs || !ref || !dL_dimgs)) || !(lambda_ssim >= 0.0) ||
      3ull * (unsigned long long)W * (unsigned long long)H >= (1ull << 32)) {
    set_error("gsr_distortion_backward: invalid argument");
    return GSR_E_INVALID_ARG;
  }
  if (lambda_ssim > 0.0 && B > 0 && (!workspace || ws_bytes < gsr_distortion_backward_workspace_bytes(H, W))) {
    set_error("gsr_distortion_backward: workspace too small (needs %zu bytes)", gsr_distortion_backward_workspace_bytes(H, W));
    return GSR_E_WORKSPACE_TOO_SMALL;
  }
  if (launch_distortion_backward(imgs, ref, B, H, W, weight, lambda_ssim, dL_dimgs, (double*)workspace,
                                 (cudaStream_t)cuda_stream) != 0) {
    set_error("gsr_distortion_backward: shared-memory opt-in failed: %s", cudaGetErrorString(cudaGetLastError()));
    return GSR_E_CUDA;
  }
  GSR_CUDA(cudaGetLastError());
  return GSR_OK;
}

int gsr_project_backward(const gsr_scene* scene, const gsr_camera* cam, float t, const float* grad_records,
                         float* g_gauss, float* g_sh_base, float* g_sh_res, float* g_cluster, void* cuda_stream) {
  if (!scene || !camera_ok(cam) || !g_cluster || (scene->impl.d.N > 0 && (!grad_records || !g_gauss || !g_sh_base || !g_sh_res))) {
    set_error("gsr_project_backward: invalid argument");
    return GSR_E_INVALID_ARG;
  }
  if (((uintptr_t)grad_records & 15u) != 0) {  // rows of 12 floats are read as three 16-byte words
    set_error("gsr_project_backward: grad_records must be 16-byte aligned");
    return GSR_E_INVALID_ARG;
  }
  const DeviceScene& D = scene->impl.d;
  if (D.V != 2 || D.affine_cov) {
    set_error("gsr_project_backward: scenes with position residual levels, per-level attribute refinements or the "
              "affine on the covariance are not covered");
    return GSR_E_INVALID_ARG;
  }
  FrameParams fp;
  make_frame(&scene->impl, cam, t, &fp);
  launch_project_backward(D, fp, grad_records, g_gauss, g_sh_base, g_sh_res, g_cluster, (cudaStream_t)cuda_stream);
  GSR_CUDA(cudaGetLastError());
  return GSR_OK;
}

int gsr_project_backward_full(const gsr_scene* scene, const gsr_camera* cam, float t, const float* grad_records,
                              float* g_gauss, float* g_sh_base, float* g_sh_res, float* g_cluster, float* g_delta,
                              float* g_attr, float* g_d_sh, void* cuda_stream) {
  if (!scene || !camera_ok(cam) || !g_cluster || (scene->impl.d.N > 0 && (!grad_records || !g_gauss || !g_sh_base || !g_sh_res))) {
    set_error("gsr_project_backward_full: invalid argument");
    return GSR_E_INVALID_ARG;
  }
  if (((uintptr_t)grad_records & 15u) != 0) {
    set_error("gsr_project_backward_full: grad_records must be 16-byte aligned");
    return GSR_E_INVALID_ARG;
  }
  const DeviceScene& D = scene->impl.d;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  FrameParams fp;
  make_frame(&scene->impl, cam, t, &fp);
  if (D.V == 2) {  // two records per Gaussian: the kernel of gsr_project_backward; no refinement has any gradient
    if (D.affine_cov) {
      set_error("gsr_project_backward_full: affine_on_covariance needs a scene with four records per Gaussian");
      return GSR_E_INVALID_ARG;
    }
    launch_project_backward(D, fp, grad_records, g_gauss, g_sh_base, g_sh_res, g_cluster, st);
    const size_t N = (size_t)D.N;
    if (g_delta && N) GSR_CUDA(cudaMemsetAsync(g_delta, 0, sizeof(float) * 6 * N, st));
    if (g_attr && N) GSR_CUDA(cudaMemsetAsync(g_attr, 0, sizeof(float) * 24 * N, st));
    if (g_d_sh && N) GSR_CUDA(cudaMemsetAsync(g_d_sh, 0, sizeof(float) * 9 * (size_t)D.K * N, st));
  } else {
    launch_project_backward4(D, fp, grad_records, g_gauss, g_sh_base, g_sh_res, g_cluster, g_delta, g_attr, g_d_sh, st);
  }
  GSR_CUDA(cudaGetLastError());
  return GSR_OK;
}

int gsr_workspace_status(const void* workspace, int64_t* keys_needed, void* cuda_stream) {
  if (!workspace) { set_error("gsr_workspace_status: NULL workspace"); return GSR_E_INVALID_ARG; }
  WsHeader h;
  GSR_CUDA(cudaMemcpyAsync(&h, workspace, sizeof(h), cudaMemcpyDeviceToHost, (cudaStream_t)cuda_stream));
  GSR_CUDA(cudaStreamSynchronize((cudaStream_t)cuda_stream));
  if (keys_needed) *keys_needed = (int64_t)h.total_keys;
  if (h.status == GSR_E_WORKSPACE_TOO_SMALL)
    set_error("key capacity %lld exceeded: the frame produced %llu keys", h.key_capacity, h.total_keys);
  else if (h.status == GSR_E_INVALID_LEVEL)
    set_error("levels contains a value outside -1..3");
  return h.status;
}

size_t gsr_distortion_workspace_bytes(int32_t B, int32_t H, int32_t W) {
  if (B < 0 || H <= 0 || W <= 0) return 0;
  const size_t tiles = (size_t)((W + kTile - 1) / kTile) * ((H + kTile - 1) / kTile);
  return align_up(sizeof(double) * (size_t)(B > 0 ? B : 1) * tiles);
}

int gsr_distortion(const float* imgs, const float* ref, int32_t B, int32_t H, int32_t W, double* mse,
                   float* psnr_db, void* workspace, size_t ws_bytes, void* cuda_stream) {
  if (B < 0 || H <= 0 || W <= 0 || (B > 0 && (!imgs || !ref || !mse)) || !workspace) {
    set_error("gsr_distortion: invalid argument");
    return GSR_E_INVALID_ARG;
  }
  if (ws_bytes < gsr_distortion_workspace_bytes(B, H, W)) {
    set_error("gsr_distortion: workspace too small");
    return GSR_E_WORKSPACE_TOO_SMALL;
  }
  launch_distortion(imgs, ref, B, H, W, (double*)workspace, mse, psnr_db, (cudaStream_t)cuda_stream);
  GSR_CUDA(cudaGetLastError());
  return GSR_OK;
}

int64_t gsr_distortion_static_max_partials(void) { return (int64_t)kStaticPartials; }

int gsr_distortion_static(const float* imgs, const float* ref, int32_t B, int32_t H, int32_t W, double* mse,
                          float* psnr_db, void* cuda_stream) {
  if (B < 0 || H <= 0 || W <= 0 || (B > 0 && (!imgs || !ref || !mse))) {
    set_error("gsr_distortion_static: invalid argument");
    return GSR_E_INVALID_ARG;
  }
  const long long tiles = (long long)((W + kTile - 1) / kTile) * (long long)((H + kTile - 1) / kTile);
  if ((long long)B * tiles > kStaticPartials) {
    set_error("gsr_distortion_static: B * tiles = %lld exceeds the built-in scratch of %lld partials "
              "(use gsr_distortion with a workspace)", (long long)B * tiles, kStaticPartials);
    return GSR_E_WORKSPACE_TOO_SMALL;
  }
  const int rc = launch_distortion_static(imgs, ref, B, H, W, mse, psnr_db, (cudaStream_t)cuda_stream);
  if (rc != 0) {
    set_error("gsr_distortion_static: cudaGetSymbolAddress failed: %s", cudaGetErrorString((cudaError_t)rc));
    return GSR_E_CUDA;
  }
  GSR_CUDA(cudaGetLastError());
  return GSR_OK;
}

static int group_utility(const double* mse, const float* psnr_db, int32_t B, const int32_t* idx_without,
                         const int32_t* idx_with, const int32_t* group_id, int32_t n_pairs, int32_t G, gsr_utility* out,
                         double* delta_mse, double* delta_db, void* cuda_stream) {
  if (n_pairs < 0 || G < 0 || (n_pairs > 0 && (!mse || !psnr_db || !idx_without || !idx_with || !group_id)) ||
      (G > 0 && !out)) {
    set_error("gsr_group_utility: invalid argument");
    return GSR_E_INVALID_ARG;
  }
  launch_group_utility(mse, psnr_db, B, idx_without, idx_with, group_id, n_pairs, G, out, delta_mse, delta_db,
                       (cudaStream_t)cuda_stream);
  GSR_CUDA(cudaGetLastError());
  return GSR_OK;
}

int gsr_group_utility(const double* mse, const float* psnr_db, const int32_t* idx_without, const int32_t* idx_with,
                      const int32_t* group_id, int32_t n_pairs, int32_t G, gsr_utility* out, double* delta_mse,
                      double* delta_db, void* cuda_stream) {
  return group_utility(mse, psnr_db, -1, idx_without, idx_with, group_id, n_pairs, G, out, delta_mse, delta_db,
                       cuda_stream);
}

int gsr_group_utility_b(const double* mse, const float* psnr_db, int32_t B, const int32_t* idx_without,
                        const int32_t* idx_with, const int32_t* group_id, int32_t n_pairs, int32_t G, gsr_utility* out,
                        double* delta_mse, double* delta_db, void* cuda_stream) {
  if (B < 0) { set_error("gsr_group_utility_b: B < 0"); return GSR_E_INVALID_ARG; }
  return group_utility(mse, psnr_db, B, idx_without, idx_with, group_id, n_pairs, G, out, delta_mse, delta_db,
                       cuda_stream);
}

int gsr_index_status(void* cuda_stream) {
  cudaStream_t st = (cudaStream_t)cuda_stream;
  int* w = device_error_word();
  if (!w) { set_error("gsr_index_status: no error word on this device"); return GSR_E_CUDA; }
  int bits = 0;
  GSR_CUDA(cudaMemcpyAsync(&bits, w, sizeof(int), cudaMemcpyDeviceToHost, st));
  GSR_CUDA(cudaMemsetAsync(w, 0, sizeof(int), st));
  GSR_CUDA(cudaStreamSynchronize(st));
  if (bits == 0) return GSR_OK;
  set_error("index out of range on the device:%s%s%s%s", (bits & kBadOrder) ? " send order entry outside [0, 4C)" : "",
            (bits & kBadPairIndex) ? " pair state index outside [0, B)" : "",
            (bits & kBadGroupId) ? " group id outside [0, G)" : "",
            (bits & kBadPrefixIndex) ? " prefix pair index outside [0, n)" : "");
  return GSR_E_INVALID_ARG;
}

int gsr_close_levels(const uint8_t* delivered_mask, int64_t n, int8_t* depth_out, uint8_t* closure_out,
                     void* cuda_stream) {
  if (n < 0 || (n > 0 && (!delivered_mask || !depth_out))) {
    set_error("gsr_close_levels: invalid argument");
    return GSR_E_INVALID_ARG;
  }
  launch_close_levels(delivered_mask, n, depth_out, closure_out, (cudaStream_t)cuda_stream);
  GSR_CUDA(cudaGetLastError());
  return GSR_OK;
}

// ------------------------------------------------------------------------------------------------
// scheduling frontier / partial-state atlas
int gsr_group_wire_bytes(const int64_t* raw_bytes, int32_t C, int64_t* wire, void* cuda_stream) {
  if (C <= 0 || C > kMaxC || !raw_bytes || !wire) { set_error("gsr_group_wire_bytes: invalid argument"); return GSR_E_INVALID_ARG; }
  launch_wire_bytes((const long long*)raw_bytes, C, (long long*)wire, (cudaStream_t)cuda_stream);
  GSR_CUDA(cudaGetLastError());
  return GSR_OK;
}

int gsr_frontier_order(const double* score, const int64_t* wire, int32_t C, int32_t policy, int32_t* order,
                       int64_t* cum_bytes, void* cuda_stream) {
  if (C <= 0 || C > kMaxC || !wire || !order || policy < GSR_POLICY_UTILITY || policy > GSR_POLICY_BYTE_GREEDY ||
      (policy == GSR_POLICY_UTILITY && !score)) {
    set_error("gsr_frontier_order: invalid argument");
    return GSR_E_INVALID_ARG;
  }
  launch_frontier_order(score, (const long long*)wire, C, policy, order, (long long*)cum_bytes,
                        (cudaStream_t)cuda_stream);
  GSR_CUDA(cudaGetLastError());
  return GSR_OK;
}

int gsr_frontier_states(const int32_t* order, const int64_t* wire, int32_t C, const int64_t* budgets, int32_t nb,
                        int8_t* levels, int64_t* used, int32_t* n_groups, void* cuda_stream) {
  if (C <= 0 || C > kMaxC || nb < 0 || !order || !wire || (nb > 0 && (!budgets || !levels))) {
    set_error("gsr_frontier_states: invalid argument");
    return GSR_E_INVALID_ARG;
  }
  launch_frontier_states(order, (const long long*)wire, C, (const long long*)budgets, nb, levels, (long long*)used,
                         n_groups, (cudaStream_t)cuda_stream);
  GSR_CUDA(cudaGetLastError());
  return GSR_OK;
}

int gsr_state_bytes(const int8_t* levels, int32_t B, int32_t C, const int64_t* wire, int64_t* bytes,
                    void* cuda_stream) {
  if (C <= 0 || C > kMaxC || B < 0 || !wire || (B > 0 && (!levels || !bytes))) {
    set_error("gsr_state_bytes: invalid argument");
    return GSR_E_INVALID_ARG;
  }
  launch_state_bytes(levels, B, C, (const long long*)wire, (long long*)bytes, (cudaStream_t)cuda_stream);
  GSR_CUDA(cudaGetLastError());
  return GSR_OK;
}

int gsr_best_state_under_budget(const float* psnr_db, const int64_t* state_bytes, int32_t B,
                                const int64_t* budgets, int32_t nb, int32_t* best, void* cuda_stream) {
  if (B < 0 || nb < 0 || (nb > 0 && (!budgets || !best)) || (B > 0 && (!psnr_db || !state_bytes))) {
    set_error("gsr_best_state_under_budget: invalid argument");
    return GSR_E_INVALID_ARG;
  }
  launch_best_under_budget(psnr_db, (const long long*)state_bytes, B, (const long long*)budgets, nb, best,
                           (cudaStream_t)cuda_stream);
  GSR_CUDA(cudaGetLastError());
  return GSR_OK;
}

// ------------------------------------------------------------------------------------------------
// richer distortion / risk reductions
int gsr_distortion_ssim(const float* imgs, const float* ref, int32_t B, int32_t H, int32_t W, const double* mse,
                        double* ssim, double* d_mix, void* workspace, size_t ws_bytes, void* cuda_stream) {
  if (B < 0 || H <= 0 || W <= 0 || (B > 0 && (!imgs || !ref || (!ssim && !d_mix))) || (d_mix && !mse) || !workspace) {
    set_error("gsr_distortion_ssim: invalid argument");
    return GSR_E_INVALID_ARG;
  }
  if (ws_bytes < gsr_distortion_workspace_bytes(B, H, W)) {
    set_error("gsr_distortion_ssim: workspace too small");
    return GSR_E_WORKSPACE_TOO_SMALL;
  }
  launch_ssim(imgs, ref, B, H, W, mse, (double*)workspace, ssim, d_mix, (cudaStream_t)cuda_stream);
  GSR_CUDA(cudaGetLastError());
  return GSR_OK;
}

int gsr_flicker(const float* imgs_t1, const float* imgs_t2, const float* ref_t1, const float* ref_t2, int32_t B,
                int32_t H, int32_t W, double* out, void* workspace, size_t ws_bytes, void* cuda_stream) {
  if (B < 0 || H <= 0 || W <= 0 || (B > 0 && (!imgs_t1 || !imgs_t2 || !ref_t1 || !ref_t2 || !out)) || !workspace) {
    set_error("gsr_flicker: invalid argument");
    return GSR_E_INVALID_ARG;
  }
  if (ws_bytes < gsr_distortion_workspace_bytes(B, H, W)) {
    set_error("gsr_flicker: workspace too small");
    return GSR_E_WORKSPACE_TOO_SMALL;
  }
  launch_flicker(imgs_t1, imgs_t2, ref_t1, ref_t2, B, H, W, (double*)workspace, out, (cudaStream_t)cuda_stream);
  GSR_CUDA(cudaGetLastError());
  return GSR_OK;
}

int gsr_risk_reduce(const void* values, int32_t dtype, int32_t n, double alpha, int32_t upper_tail, gsr_risk* out,
                    void* cuda_stream) {
  if (n < 0 || (n > 0 && !values) || !out || (dtype != 0 && dtype != 1) || !(alpha > 0.0) || alpha > 1.0) {
    set_error("gsr_risk_reduce: invalid argument");
    return GSR_E_INVALID_ARG;
  }
  launch_risk_reduce(values, dtype, n, alpha, upper_tail != 0, out, (cudaStream_t)cuda_stream);
  GSR_CUDA(cudaGetLastError());
  return GSR_OK;
}

static int prefix_monotonicity(const double* d, int32_t n, const int32_t* idx_prev, const int32_t* idx_next,
                               int32_t n_pairs, double* m_out, int32_t* violations, void* cuda_stream) {
  if (n_pairs < 0 || (n_pairs > 0 && (!d || !idx_prev || !idx_next)) || (!m_out && !violations)) {
    set_error("gsr_prefix_monotonicity: invalid argument");
    return GSR_E_INVALID_ARG;
  }
  launch_prefix_monotonicity(d, n, idx_prev, idx_next, n_pairs, m_out, violations, (cudaStream_t)cuda_stream);
  GSR_CUDA(cudaGetLastError());
  return GSR_OK;
}

int gsr_prefix_monotonicity(const double* d, const int32_t* idx_prev, const int32_t* idx_next, int32_t n_pairs,
                            double* m_out, int32_t* violations, void* cuda_stream) {
  return prefix_monotonicity(d, -1, idx_prev, idx_next, n_pairs, m_out, violations, cuda_stream);
}

int gsr_prefix_monotonicity_n(const double* d, int32_t n, const int32_t* idx_prev, const int32_t* idx_next,
                              int32_t n_pairs, double* m_out, int32_t* violations, void* cuda_stream) {
  if (n < 0) { set_error("gsr_prefix_monotonicity_n: n < 0"); return GSR_E_INVALID_ARG; }
  return prefix_monotonicity(d, n, idx_prev, idx_next, n_pairs, m_out, violations, cuda_stream);
}

// ------------------------------------------------------------------------------------------------
// delivery-mask sampler
size_t gsr_delivery_workspace_bytes(int32_t C) { return C > 0 ? align_up(delivery_workspace_bytes(C)) : 0; }

int gsr_sample_delivery(const int64_t* raw_bytes, const int32_t* order, int32_t C, const gsr_loss_model* model,
                        const int32_t* packet_budget, int32_t W, int32_t world0, uint8_t* mask, int8_t* levels,
                        void* workspace, size_t ws_bytes, void* cuda_stream) {
  if (C <= 0 || C > kMaxC || W < 0 || world0 < 0 || !raw_bytes || !order || !model || !workspace ||
      (W > 0 && !mask)) {
    set_error("gsr_sample_delivery: invalid argument");
    return GSR_E_INVALID_ARG;
  }
  const double ps[5] = {model->p_iid, model->p_gb, model->p_bg, model->e_good, model->e_bad};
  for (double p : ps)
    if (!(p >= 0.0 && p <= 1.0)) { set_error("gsr_sample_delivery: probabilities must be in [0, 1]"); return GSR_E_INVALID_ARG; }
  if (ws_bytes < delivery_workspace_bytes(C)) { set_error("gsr_sample_delivery: workspace too small"); return GSR_E_WORKSPACE_TOO_SMALL; }
  launch_sample_delivery((const long long*)raw_bytes, order, C, *model, packet_budget, W, world0, mask, levels,
                         (long long*)workspace, (cudaStream_t)cuda_stream);
  GSR_CUDA(cudaGetLastError());
  return GSR_OK;
}

// ------------------------------------------------------------------------------------------------
// host-buffer convenience call (end-to-end measurement)
struct FrameCarve {
  size_t o_render, o_levels, o_full, o_ref, o_mse, o_psnr, o_pairs, o_util, o_out, o_refmse, total;
};

static FrameCarve carve_frame(const gsr_scene* scene, const gsr_camera* cam, int32_t B, int32_t n_pairs, int32_t G,
                              int want_images) {
  FrameCarve f;
  size_t off = 0;
  auto take = [&](size_t bytes) { size_t o = off; off += align_up(bytes); return o; };
  const size_t P3 = (size_t)cam->W * cam->H * 3;
  f.o_render = take(gsr_workspace_bytes(scene, cam, B > 1 ? B : 1));
  f.o_levels = take((size_t)B * scene->impl.d.C);
  f.o_full = take((size_t)scene->impl.d.C);
  f.o_ref = take(sizeof(float) * P3);
  f.o_mse = take(sizeof(double) * (size_t)(B + 1));
  f.o_psnr = take(sizeof(float) * (size_t)(B + 1));
  f.o_pairs = take(sizeof(int32_t) * 3 * (size_t)(n_pairs > 0 ? n_pairs : 1));
  f.o_util = take(sizeof(gsr_utility) * (size_t)(G > 0 ? G : 1));
  f.o_out = take(want_images ? sizeof(float) * P3 * (size_t)B : 0);
  f.o_refmse = take(64);
  f.total = off;
  return f;
}

size_t gsr_frame_workspace_bytes(const gsr_scene* scene, const gsr_camera* cam, int32_t B, int32_t n_pairs,
                                 int32_t G, int32_t want_images) {
  if (!scene || !camera_ok(cam) || B < 0 || n_pairs < 0 || G < 0) return 0;
  return carve_frame(scene, cam, B, n_pairs, G, want_images).total;
}

int gsr_utility_frame_host(const gsr_scene* scene, const gsr_camera* cam, float t, const int8_t* levels, int32_t B,
                           const int32_t* idx_without, const int32_t* idx_with, const int32_t* group_id,
                           int32_t n_pairs, int32_t G, double* mse, float* psnr_db, gsr_utility* util,
                           int32_t materialise_images, float* out_host, void* workspace, size_t ws_bytes,
                           void* cuda_stream) {
  if (!scene || !camera_ok(cam) || B <= 0 || !levels || !mse || !psnr_db || !workspace || n_pairs < 0 || G < 0 ||
      (n_pairs > 0 && (!idx_without || !idx_with || !group_id)) || (G > 0 && !util)) {
    set_error("gsr_utility_frame_host: invalid argument");
    return GSR_E_INVALID_ARG;
  }
  for (int32_t p = 0; p < n_pairs; ++p) {  // the pair lists are on the host here: refuse bad entries before any work
    if (idx_without[p] < 0 || idx_without[p] >= B || idx_with[p] < 0 || idx_with[p] >= B) {
      set_error("gsr_utility_frame_host: pair %d has a state index outside [0, %d)", p, B);
      return GSR_E_INVALID_ARG;
    }
    if (group_id[p] < 0 || group_id[p] >= G) {
      set_error("gsr_utility_frame_host: pair %d has group id %d outside [0, %d)", p, group_id[p], G);
      return GSR_E_INVALID_ARG;
    }
  }
  if (out_host) materialise_images = 1;
  const FrameCarve f = carve_frame(scene, cam, B, n_pairs, G, materialise_images);
  if (ws_bytes < f.total) { set_error("gsr_utility_frame_host: workspace too small"); return GSR_E_WORKSPACE_TOO_SMALL; }
  cudaStream_t st = (cudaStream_t)cuda_stream;
  char* base = (char*)workspace;
  const int C = scene->impl.d.C;
  int8_t* d_levels = (int8_t*)(base + f.o_levels);
  int8_t* d_full = (int8_t*)(base + f.o_full);
  float* d_ref = (float*)(base + f.o_ref);
  double* d_mse = (double*)(base + f.o_mse);
  float* d_psnr = (float*)(base + f.o_psnr);
  int32_t* d_pairs = (int32_t*)(base + f.o_pairs);
  gsr_utility* d_util = (gsr_utility*)(base + f.o_util);
  float* d_out = materialise_images ? (float*)(base + f.o_out) : nullptr;
  void* rws = base + f.o_render;
  const size_t rws_bytes = gsr_workspace_bytes(scene, cam, B > 1 ? B : 1);
  GSR_CUDA(cudaMemcpyAsync(d_levels, levels, (size_t)B * C, cudaMemcpyHostToDevice, st));
  GSR_CUDA(cudaMemsetAsync(d_full, 3, (size_t)C, st));
  if (n_pairs > 0) {
    GSR_CUDA(cudaMemcpyAsync(d_pairs, idx_without, sizeof(int32_t) * n_pairs, cudaMemcpyHostToDevice, st));
    GSR_CUDA(cudaMemcpyAsync(d_pairs + n_pairs, idx_with, sizeof(int32_t) * n_pairs, cudaMemcpyHostToDevice, st));
    GSR_CUDA(cudaMemcpyAsync(d_pairs + 2 * (size_t)n_pairs, group_id, sizeof(int32_t) * n_pairs, cudaMemcpyHostToDevice, st));
  }
  // reference = the full state (reading A16) and the batch with fused distortion, one projection + sort
  int rc = gsr_render_states_vs_full(scene, cam, t, d_levels, B, d_out, d_ref, d_mse, d_psnr, rws, rws_bytes, st);
  if (rc != GSR_OK) return rc;
  if (G > 0) {
    rc = gsr_group_utility_b(d_mse, d_psnr, B, d_pairs, d_pairs + n_pairs, d_pairs + 2 * (size_t)n_pairs, n_pairs, G,
                             d_util, nullptr, nullptr, st);
    if (rc != GSR_OK) return rc;
  }
  GSR_CUDA(cudaMemcpyAsync(mse, d_mse, sizeof(double) * B, cudaMemcpyDeviceToHost, st));
  GSR_CUDA(cudaMemcpyAsync(psnr_db, d_psnr, sizeof(float) * B, cudaMemcpyDeviceToHost, st));
  if (G > 0) GSR_CUDA(cudaMemcpyAsync(util, d_util, sizeof(gsr_utility) * G, cudaMemcpyDeviceToHost, st));
  if (out_host)
    GSR_CUDA(cudaMemcpyAsync(out_host, d_out, sizeof(float) * 3 * (size_t)cam->W * cam->H * B, cudaMemcpyDeviceToHost, st));
  return gsr_workspace_status(rws, nullptr, st);
}

// ------------------------------------------------------------------------------------------------
// debug / parity exports
static int ws_from(const gsr_scene* scene, const void* workspace, Workspace* ws, WsHeader* h, cudaStream_t st) {
  if (!scene || !workspace) { set_error("debug: NULL argument"); return GSR_E_INVALID_ARG; }
  GSR_CUDA(cudaMemcpyAsync(h, workspace, sizeof(*h), cudaMemcpyDeviceToHost, st));
  GSR_CUDA(cudaStreamSynchronize(st));
  if (h->N != scene->impl.d.N || h->C != scene->impl.d.C) { set_error("debug: workspace does not belong to this scene"); return GSR_E_INVALID_ARG; }
  carve_workspace(ws, const_cast<void*>(workspace), rec_half(scene->impl.d), h->C, h->B, h->TX * h->TY, h->key_capacity);
  return GSR_OK;
}

int gsr_debug_projection(const gsr_scene* scene, const void* workspace, uint8_t* valid, int32_t* radius,
                         int32_t* rect, uint32_t* depth_bits, int32_t* count, float* mean2d, float* conic,
                         float* rgb_base, float* rgb_res, void* cuda_stream) {
  cudaStream_t st = (cudaStream_t)cuda_stream;
  Workspace ws; WsHeader h;
  int rc = ws_from(scene, workspace, &ws, &h, st);
  if (rc != GSR_OK) return rc;
  const size_t n = (size_t)scene->impl.d.V * (size_t)h.N;
  std::vector<float4> r0(n), r1(n), c0(n), c1(n);
  std::vector<int32_t> rad(n);
  std::vector<uint2> rc4(n);
  std::vector<uint32_t> db(n), cnt(n);
  GSR_CUDA(cudaMemcpy(r0.data(), ws.r0, sizeof(float4) * n, cudaMemcpyDeviceToHost));
  GSR_CUDA(cudaMemcpy(r1.data(), ws.r1, sizeof(float4) * n, cudaMemcpyDeviceToHost));
  GSR_CUDA(cudaMemcpy(c0.data(), ws.rc0, sizeof(float4) * n, cudaMemcpyDeviceToHost));
  GSR_CUDA(cudaMemcpy(c1.data(), ws.rc1, sizeof(float4) * n, cudaMemcpyDeviceToHost));
  GSR_CUDA(cudaMemcpy(rad.data(), ws.radius, sizeof(int32_t) * n, cudaMemcpyDeviceToHost));
  GSR_CUDA(cudaMemcpy(rc4.data(), ws.rect, sizeof(uint2) * n, cudaMemcpyDeviceToHost));
  GSR_CUDA(cudaMemcpy(db.data(), ws.depth_bits, sizeof(uint32_t) * n, cudaMemcpyDeviceToHost));
  GSR_CUDA(cudaMemcpy(cnt.data(), ws.count, sizeof(uint32_t) * n, cudaMemcpyDeviceToHost));
  for (size_t r = 0; r < n; ++r) {
    if (valid) valid[r] = cnt[r] > 0;
    if (radius) radius[r] = rad[r];
    if (rect) {
      rect[4 * r + 0] = rc4[r].x & 0xFFFF; rect[4 * r + 1] = rc4[r].x >> 16;
      rect[4 * r + 2] = rc4[r].y & 0xFFFF; rect[4 * r + 3] = rc4[r].y >> 16;
    }
    if (depth_bits) depth_bits[r] = db[r];
    if (count) count[r] = (int32_t)cnt[r];
    if (mean2d) { mean2d[2 * r] = r0[r].x; mean2d[2 * r + 1] = r0[r].y; }
    if (conic) { conic[3 * r] = r0[r].z; conic[3 * r + 1] = r0[r].w; conic[3 * r + 2] = r1[r].x; }
    if (rgb_base) { rgb_base[3 * r] = c0[r].x; rgb_base[3 * r + 1] = c0[r].y; rgb_base[3 * r + 2] = c0[r].z; }
    if (rgb_res) { rgb_res[3 * r] = c1[r].x; rgb_res[3 * r + 1] = c1[r].y; rgb_res[3 * r + 2] = c1[r].z; }
  }
  return GSR_OK;
}

int gsr_debug_keys(const gsr_scene* scene, const void* workspace, int32_t b, int64_t cap, uint32_t* tile,
                   uint32_t* depth_bits, int32_t* gaussian, int64_t* n_keys, void* cuda_stream) {
  cudaStream_t st = (cudaStream_t)cuda_stream;
  Workspace ws; WsHeader h;
  int rc = ws_from(scene, workspace, &ws, &h, st);
  if (rc != GSR_OK) return rc;
  if (b < 0 || b >= h.B || cap < 0 || !n_keys) { set_error("gsr_debug_keys: invalid argument"); return GSR_E_INVALID_ARG; }
  const size_t m = (size_t)(cap > 0 ? cap : 1);
  // one allocation for the counter and the three key columns, released on every exit path
  struct DevBuf {
    char* p = nullptr;
    ~DevBuf() { if (p) cudaFree(p); }
  } buf;
  GSR_CUDA(cudaMalloc(&buf.p, 8 + 12 * m));
  unsigned long long* d_n = (unsigned long long*)buf.p;
  uint32_t* d_tile = (uint32_t*)(buf.p + 8);
  uint32_t* d_db = d_tile + m;
  int32_t* d_gi = (int32_t*)(d_db + m);
  launch_filter_keys(scene->impl.d, ws, b, d_tile, d_db, d_gi, d_n, cap, st);
  unsigned long long n = 0;
  GSR_CUDA(cudaMemcpyAsync(&n, d_n, 8, cudaMemcpyDeviceToHost, st));
  GSR_CUDA(cudaStreamSynchronize(st));
  const size_t ncopy = (size_t)((long long)n < cap ? (long long)n : cap);
  if (ncopy) {
    if (tile) GSR_CUDA(cudaMemcpy(tile, d_tile, 4 * ncopy, cudaMemcpyDeviceToHost));
    if (depth_bits) GSR_CUDA(cudaMemcpy(depth_bits, d_db, 4 * ncopy, cudaMemcpyDeviceToHost));
    if (gaussian) GSR_CUDA(cudaMemcpy(gaussian, d_gi, 4 * ncopy, cudaMemcpyDeviceToHost));
  }
  *n_keys = (int64_t)n;
  return GSR_OK;
}

int gsr_debug_state_counts(const gsr_scene* scene, const void* workspace, int64_t* counts, void* cuda_stream) {
  cudaStream_t st = (cudaStream_t)cuda_stream;
  Workspace ws; WsHeader h;
  int rc = ws_from(scene, workspace, &ws, &h, st);
  if (rc != GSR_OK) return rc;
  if (!counts) { set_error("gsr_debug_state_counts: NULL counts"); return GSR_E_INVALID_ARG; }
  launch_state_counts(scene->impl.d, ws, h.B, st);
  GSR_CUDA(cudaMemcpyAsync(counts, ws.state_counts, sizeof(long long) * (size_t)h.B, cudaMemcpyDeviceToHost, st));
  GSR_CUDA(cudaStreamSynchronize(st));
  return GSR_OK;
}

int gsr_debug_pair_counts(const gsr_scene* scene, const void* workspace, int64_t* counts3, void* cuda_stream) {
  cudaStream_t st = (cudaStream_t)cuda_stream;
  Workspace ws; WsHeader h;
  int rc = ws_from(scene, workspace, &ws, &h, st);
  if (rc != GSR_OK) return rc;
  if (!counts3) { set_error("gsr_debug_pair_counts: NULL counts"); return GSR_E_INVALID_ARG; }
  unsigned long long* d_c = nullptr;
  GSR_CUDA(cudaMalloc(&d_c, 24));
  GSR_CUDA(cudaMemsetAsync(d_c, 0, 24, st));
  FrameParams fp;
  memset(&fp, 0, sizeof(fp));
  fp.W = h.W; fp.H = h.H; fp.TX = h.TX; fp.TY = h.TY;
  launch_composite_count(scene->impl.d, fp, ws, ws.depth, h.B, d_c, st);
  unsigned long long c[3];
  GSR_CUDA(cudaMemcpyAsync(c, d_c, 24, cudaMemcpyDeviceToHost, st));
  GSR_CUDA(cudaStreamSynchronize(st));
  cudaFree(d_c);
  for (int k = 0; k < 3; ++k) counts3[k] = (int64_t)c[k];
  return GSR_OK;
}

int gsr_debug_closure(const gsr_scene* scene, const void* workspace, int8_t* depth, void* cuda_stream) {
  cudaStream_t st = (cudaStream_t)cuda_stream;
  Workspace ws; WsHeader h;
  int rc = ws_from(scene, workspace, &ws, &h, st);
  if (rc != GSR_OK) return rc;
  if (!depth) { set_error("gsr_debug_closure: NULL depth"); return GSR_E_INVALID_ARG; }
  GSR_CUDA(cudaMemcpyAsync(depth, ws.depth, (size_t)h.B * h.C, cudaMemcpyDeviceToHost, st));
  GSR_CUDA(cudaStreamSynchronize(st));
  return GSR_OK;
}

}  // extern "C"
