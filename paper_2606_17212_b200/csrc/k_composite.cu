// k_composite.cu — host side of stage a4 (+ fused a5): launch of the quadrant compositor (k_composite_q.cu) per
// chunk of states, the tile-level state dedup in front of it, the unfused distortion kernels of gsr_distortion
// (same pixel -> thread mapping and the same reduction tree as the fused path: reduce.cuh), launch bookkeeping,
// optional CUDA-event timing of the compositing launches and the FP32 peak measurement.
#include <atomic>
#include <mutex>
#include <thread>

#include "composite_common.cuh"
#include "gsr_internal.h"
#include "reduce.cuh"

namespace gsr {

// ------------------------------------------------------------------------------------------------
// gsr_distortion (unfused): same pixel->thread mapping and the same tree as the fused path
__global__ void __launch_bounds__(kTilePix) k_distortion_tiles(const float* __restrict__ imgs,
                                                               const float* __restrict__ ref, int W, int H,
                                                               int TX, int tiles, double* __restrict__ part) {
  __shared__ double s_red[8];
  const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
  const int tile = blockIdx.x, b = blockIdx.y;
  const int x = (tile % TX) * kTile + 8 * (w & 1) + (lane & 7), y = (tile / TX) * kTile + 4 * (w >> 1) + (lane >> 3);
  float e = 0.0f;
  if (x < W && y < H) {
    const size_t p = ((size_t)y * W + x) * 3;
    const float* ip = imgs + (size_t)b * H * W * 3 + p;
    e = pixel_sq_err(ip[0], ip[1], ip[2], __ldg(ref + p), __ldg(ref + p + 1), __ldg(ref + p + 2));
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

// one warp per state: tiles in index order (lane-strided), then the butterfly; MSE and PSNR
__global__ void __launch_bounds__(128) k_distortion_finalize(const double* __restrict__ part, int B, int tiles,
                                                             double inv_n, double* __restrict__ mse,
                                                             float* __restrict__ psnr) {
  const int b = blockIdx.x * 4 + (threadIdx.x >> 5), lane = threadIdx.x & 31;
  if (b >= B) return;
  double acc = 0.0;
  for (int k = lane; k < tiles; k += 32) acc += part[(size_t)b * tiles + k];
  acc = warp_sum_butterfly(acc);
  if (lane == 0) {
    const double m = acc * inv_n;
    mse[b] = m;
    if (psnr) psnr[b] = (float)(-10.0 * log10(m > 1e-10 ? m : 1e-10));
  }
}

void launch_distortion_finalize(const double* part, int32_t B, int32_t tiles, int64_t n_values, double* mse,
                                float* psnr, cudaStream_t st) {
  if (B == 0) return;
  k_distortion_finalize<<<(B + 3) / 4, 128, 0, st>>>(part, B, tiles, 1.0 / (double)n_values, mse, psnr);
}

void launch_distortion(const float* imgs, const float* ref, int32_t B, int32_t H, int32_t W, double* part,
                       double* mse, float* psnr, cudaStream_t st) {
  if (B == 0) return;
  const int TX = (W + kTile - 1) / kTile, TY = (H + kTile - 1) / kTile, tiles = TX * TY;
  for (int b0 = 0; b0 < B; b0 += 65535) {  // gridDim.y limit
    const int nb = B - b0 < 65535 ? B - b0 : 65535;
    k_distortion_tiles<<<dim3(tiles, nb), kTilePix, 0, st>>>(imgs + (size_t)b0 * H * W * 3, ref, W, H, TX, tiles,
                                                            part + (size_t)b0 * tiles);
  }
  launch_distortion_finalize(part, B, tiles, (int64_t)3 * W * H, mse, psnr, st);
}

// ------------------------------------------------------------------------------------------------
// launch bookkeeping: kernel-launch counter and optional CUDA-event timing of the compositing kernel
static std::atomic<unsigned long long> g_launches{0};  // calls may come from several host threads (one stream each)
void count_launches(int n) { g_launches.fetch_add((unsigned long long)n, std::memory_order_relaxed); }
unsigned long long launches_total() { return g_launches.load(std::memory_order_relaxed); }

// Options (gsr_set_option).  The two that steer launches belong to the CALLING HOST THREAD: a thread that sets
// them changes its own later calls only, never a launch another thread is preparing.
thread_local int g_state_block = 0;  // S; 0 = default (k_composite_q.cu); experiments: 1, 4..8, 16
thread_local int g_dedup = 1;        // tile-level state dedup on / off
// "profile" is process-wide and owned by the thread that switched it on: only that thread's calls record events
// (the event arrays below are not synchronised), calls of other threads run unprofiled.
std::atomic<int> g_profile{0};
std::thread::id g_profile_owner;
bool profiling_here() { return g_profile.load(std::memory_order_acquire) != 0 && std::this_thread::get_id() == g_profile_owner; }
constexpr int kMaxProfEvents = 8192;
static cudaEvent_t g_ev[kMaxProfEvents][2];
static int g_ev_created = 0, g_ev_used = 0;

void profile_reset() { g_ev_used = 0; }
// sum of k_composite durations (ms) and launches recorded since the last reset; synchronises the events
int profile_read(double* ms, int* n) {
  double tot = 0;
  for (int k = 0; k < g_ev_used; ++k) {
    float e = 0;
    if (cudaEventSynchronize(g_ev[k][1]) != cudaSuccess) return -1;
    if (cudaEventElapsedTime(&e, g_ev[k][0], g_ev[k][1]) != cudaSuccess) return -1;
    tot += e;
  }
  *ms = tot;
  *n = g_ev_used;
  return 0;
}

// optional CUDA events around a compositing launch (gsr_set_option("profile", 1))
static int profile_begin(cudaStream_t st) {
  int slot = -1;
  if (profiling_here() && g_ev_used < kMaxProfEvents) {
    slot = g_ev_used++;
    while (g_ev_created <= slot) {
      cudaEventCreate(&g_ev[g_ev_created][0]);
      cudaEventCreate(&g_ev[g_ev_created][1]);
      ++g_ev_created;
    }
    cudaEventRecord(g_ev[slot][0], st);
  }
  return slot;
}
static void profile_end(int slot, cudaStream_t st) {
  if (slot >= 0) cudaEventRecord(g_ev[slot][1], st);
}

static CompositeArgs make_args(const DeviceScene& sc, const FrameParams& fp, Workspace& ws, const int8_t* depth_rows,
                               int32_t B) {
  CompositeArgs a;
  a.depth = depth_rows;
  a.B = B; a.C = sc.C;
  a.W = fp.W; a.H = fp.H; a.TX = fp.TX; a.tiles = fp.TX * fp.TY;
  a.bg[0] = fp.bg[0]; a.bg[1] = fp.bg[1]; a.bg[2] = fp.bg[2];
  a.out = nullptr; a.ref = nullptr; a.counts = nullptr;
  a.uorder = nullptr; a.upos = nullptr; a.n_unique = nullptr;
  a.rec = ws.rec; a.qlist = ws.qlist; a.qrange = ws.qrange; a.sse_blk = ws.sse_blk;
  a.work_counter = ws.work_counter; a.n_items = 0;
  return a;
}

template <bool COUNT>
static void dispatch_composite(CompositeArgs& a, cudaStream_t st) {
  const int slot = COUNT ? -1 : profile_begin(st);
  launch_composite_q(a, g_state_block, COUNT, st);
  profile_end(slot, st);
  count_launches(1);
}

// Batches larger than the in-CTA signature sort of k_tile_dedup can hold (kDedupMaxStates) are composited in
// equal chunks of states; a state's pixels do not depend on what it is batched with, so this is invisible.
constexpr int kDedupMaxStates = 8192;

static int chunk_states(int32_t B) {
  if (!g_dedup || B <= kDedupMaxStates) return B;
  const int n_chunks = (B + kDedupMaxStates - 1) / kDedupMaxStates;
  return (B + n_chunks - 1) / n_chunks;
}

void launch_composite(const DeviceScene& sc, const FrameParams& fp, Workspace& ws, const int8_t* depth_rows,
                      int32_t B, float* out, const float* ref, double* mse, float* psnr, cudaStream_t st) {
  if (B == 0) return;
  const int tiles = fp.TX * fp.TY;
  const size_t img = (size_t)fp.H * fp.W * 3;
  const int step = chunk_states(B);
  for (int b0 = 0; b0 < B; b0 += step) {
    const int nb = B - b0 < step ? B - b0 : step;
    const int8_t* rows = depth_rows + (size_t)b0 * sc.C;
    CompositeArgs a = make_args(sc, fp, ws, rows, nb);
    a.out = out ? out + (size_t)b0 * img : nullptr;
    a.ref = ref;
    a.sse_blk = ws.sse_blk + (size_t)b0 * tiles * 8;
    if (g_dedup && launch_tile_dedup(sc, fp, ws, rows, nb, st)) {
      a.uorder = ws.uorder; a.upos = ws.upos; a.n_unique = ws.n_unique;
    }
    dispatch_composite<false>(a, st);
  }
  if (ref) launch_distortion_finalize_blk(ws.sse_blk, B, tiles, (int64_t)3 * fp.W * fp.H, mse, psnr, st);
}

void launch_composite_count(const DeviceScene& sc, const FrameParams& fp, Workspace& ws, const int8_t* depth_rows,
                            int32_t B, unsigned long long* counts, cudaStream_t st) {
  if (B == 0) return;
  const int step = chunk_states(B);
  for (int b0 = 0; b0 < B; b0 += step) {
    const int nb = B - b0 < step ? B - b0 : step;
    const int8_t* rows = depth_rows + (size_t)b0 * sc.C;
    CompositeArgs a = make_args(sc, fp, ws, rows, nb);
    a.counts = counts;
    if (g_dedup && launch_tile_dedup(sc, fp, ws, rows, nb, st)) {
      a.uorder = ws.uorder; a.upos = ws.upos; a.n_unique = ws.n_unique;
    }
    dispatch_composite<true>(a, st);
  }
}

// ------------------------------------------------------------------------------------------------
// FP32 FMA-pipe peak of this device, measured: 8 independent FFMA chains per thread, 2 x 512-thread
// CTAs per SM.  Denominator of the compositing kernel's roofline.
__global__ void __launch_bounds__(512) k_ffma_peak(float* sink, int iters, float a, float b) {
  float x0 = threadIdx.x, x1 = x0 + 1, x2 = x0 + 2, x3 = x0 + 3, x4 = x0 + 4, x5 = x0 + 5, x6 = x0 + 6, x7 = x0 + 7;
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int u = 0; u < 16; ++u) {
      x0 = fmaf(x0, a, b); x1 = fmaf(x1, a, b); x2 = fmaf(x2, a, b); x3 = fmaf(x3, a, b);
      x4 = fmaf(x4, a, b); x5 = fmaf(x5, a, b); x6 = fmaf(x6, a, b); x7 = fmaf(x7, a, b);
    }
  }
  float s = x0 + x1 + x2 + x3 + x4 + x5 + x6 + x7;
  if (s == 12345.678f) sink[0] = s;
}

int measure_ffma_peak(int num_sms, double* tflops, cudaStream_t st) {
  float* sink = nullptr;
  if (cudaMalloc(&sink, 4) != cudaSuccess) return -1;
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0); cudaEventCreate(&e1);
  const int iters = 4096, grid = num_sms * 4;
  k_ffma_peak<<<grid, 512, 0, st>>>(sink, 64, 0.999f, 0.001f);  // warm-up
  double best = 0;
  for (int rep = 0; rep < 5; ++rep) {
    cudaEventRecord(e0, st);
    k_ffma_peak<<<grid, 512, 0, st>>>(sink, iters, 0.999f, 0.001f);
    cudaEventRecord(e1, st);
    if (cudaEventSynchronize(e1) != cudaSuccess) { cudaFree(sink); return -1; }
    float ms = 0;
    cudaEventElapsedTime(&ms, e0, e1);
    const double flop = 2.0 * 8 * 16 * (double)iters * 512.0 * grid;
    const double tf = flop / (ms * 1e-3) / 1e12;
    if (tf > best) best = tf;
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  cudaFree(sink);
  *tflops = best;
  return 0;
}

// ------------------------------------------------------------------------------------------------
// gsr_distortion_static: gsr_distortion for callers that may not allocate (CUDA graph capture, serving loops,
// harnesses that forbid cudaMalloc).  The per-(state, tile) partials live in a file-scope device array instead of a
// caller-provided workspace: kStaticPartials doubles = 8 MiB, held by every GPU that loads the library until exit.
// In HOST code the array's name is a host-side stand-in, not a device address: the address is asked for once per
// device (that device current) with cudaGetSymbolAddress and handed to the kernels.  Every call on a device shares
// the array: k_distortion_tiles writes every partial the finalize step reads, so nothing has to start at zero and a
// previous call's contents are harmless — but two calls that overlap on the GPU (different streams) race.
static __device__ __align__(256) double g_static_partials[kStaticPartials];

static std::mutex g_static_mu;
static double* g_static_ptr[64] = {};  // per device ordinal

// 0 and *out = the device address of g_static_partials on the CURRENT device, or the CUDA error code
static int static_partials_address(double** out) {
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return (int)e;
  if (dev < 0 || dev >= 64) return (int)cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lock(g_static_mu);
  if (!g_static_ptr[dev]) {
    void* p = nullptr;
    e = cudaGetSymbolAddress(&p, g_static_partials);
    if (e != cudaSuccess) return (int)e;
    g_static_ptr[dev] = (double*)p;
  }
  *out = g_static_ptr[dev];
  return 0;
}

// Same kernels, same reduction tree as launch_distortion.  Returns 0, or a CUDA error code from the set-up.
int launch_distortion_static(const float* imgs, const float* ref, int32_t B, int32_t H, int32_t W, double* mse,
                             float* psnr, cudaStream_t st) {
  if (B == 0) return 0;
  double* part = nullptr;
  const int rc = static_partials_address(&part);
  if (rc != 0) return rc;
  const int TX = (W + kTile - 1) / kTile, TY = (H + kTile - 1) / kTile, tiles = TX * TY;
  for (int b0 = 0; b0 < B; b0 += 65535) {  // gridDim.y limit
    const int nb = B - b0 < 65535 ? B - b0 : 65535;
    k_distortion_tiles<<<dim3(tiles, nb), kTilePix, 0, st>>>(imgs + (size_t)b0 * H * W * 3, ref, W, H, TX, tiles,
                                                            part + (size_t)b0 * tiles);
  }
  launch_distortion_finalize(part, B, tiles, (int64_t)3 * W * H, mse, psnr, st);
  return 0;
}

}  // namespace gsr
