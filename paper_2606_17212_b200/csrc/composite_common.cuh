// composite_common.cuh — shared by k_composite.cu (host side) and k_composite_q.cu (kernel): the argument block,
// explicit shared-memory accessors and the constants of DESIGN.md §3.5.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace gsr {

struct CompositeArgs {
  const float4* rec;     // [4 * records] packed 64-byte records (k_project)
  const uint2* qlist;    // per (tile, 8x8 quadrant) render lists of {record id, meta} (tile_render_lists in k_tile_sort)
  const uint2* qrange;   // [tiles * 4] start, end into qlist
  const int8_t* depth;   // [B, C] validated delivered depths
  int32_t B, C, nsb;
  int32_t W, H, TX, tiles;
  uint32_t n_items;        // work items of the launch = tiles * 4 * nsb
  uint32_t* work_counter;  // next work item (zeroed before the launch)
  float bg[3];
  float* out;          // [B,H,W,3] or nullptr
  const float* ref;    // [H,W,3] or nullptr
  double* sse_blk;     // [B, tiles, 8] per-(state, tile, 8x4 block) squared-error partials
  unsigned long long* counts;  // instrumented run only: [3] (see launch_composite_count)
  const uint32_t *uorder, *upos, *n_unique;  // tile-level state dedup (k_tile_dedup); n_unique == nullptr: off
};

__device__ __forceinline__ float4 lds128(uint32_t addr) {
  float4 v;
  asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr));
  return v;
}

__device__ __forceinline__ uint2 lds64(uint32_t addr) {
  uint2 v;
  asm volatile("ld.shared.v2.u32 {%0, %1}, [%2];" : "=r"(v.x), "=r"(v.y) : "r"(addr));
  return v;
}
__device__ __forceinline__ uint32_t lds32(uint32_t addr) {
  uint32_t v;
  asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(addr));
  return v;
}
__device__ __forceinline__ uint32_t lds16(uint32_t addr) {
  uint32_t v;
  asm volatile("ld.shared.u16 %0, [%1];" : "=r"(v) : "r"(addr));
  return v;
}
__device__ __forceinline__ void sts32(uint32_t addr, uint32_t v) {
  asm volatile("st.shared.u32 [%0], %1;" ::"r"(addr), "r"(v) : "memory");
}
__device__ __forceinline__ void sts16(uint32_t addr, uint32_t v) {
  asm volatile("st.shared.u16 [%0], %1;" ::"r"(addr), "h"((unsigned short)v) : "memory");
}
__device__ __forceinline__ float2 lds64f(uint32_t addr) {
  float2 v;
  asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "r"(addr));
  return v;
}

__device__ __forceinline__ float ex2_approx_ftz(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}

constexpr float kTStop = 1e-4f;     // reading A11
constexpr float kAlphaCap = 0.99f;  // reading A11


// ---- packed FP32 (Blackwell fma/mul/add.rn.f32x2: SASS FFMA2 / FMUL2 / FADD2), two pixels per lane
typedef unsigned long long f32x2;
constexpr float kTScale = 1099511627776.0f;                       // 2^40
constexpr float kTStopScaled = 109951160.0f;                      // 1e-4f * 2^40 (0x4CD1B717)
constexpr float kInvTScale = 9.094947017729282379150390625e-13f;  // 2^-40

__device__ __forceinline__ f32x2 pack2(float lo, float hi) {
  f32x2 r;
  asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
  return r;
}
__device__ __forceinline__ void unpack2(f32x2 v, float& lo, float& hi) {
  asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ f32x2 add2(f32x2 a, f32x2 b) {
  f32x2 r;
  asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
  return r;
}
__device__ __forceinline__ f32x2 mul2(f32x2 a, f32x2 b) {
  f32x2 r;
  asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
  return r;
}
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c) {
  f32x2 r;
  asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
  return r;
}

// ---- cp.async staging of 64-byte records
__device__ __forceinline__ void cp_async16(uint32_t saddr, const void* gptr) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(saddr), "l"(gptr) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() {
  asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory");
}

constexpr int kChunk = 32;  // list entries staged per round: one per lane

}  // namespace gsr
