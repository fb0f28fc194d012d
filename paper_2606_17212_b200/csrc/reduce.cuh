// reduce.cuh — the ONE canonical reduction tree of the per-state squared error.
// Used by the fused path (inside the compositing kernel) and by gsr_distortion, so that both give
// bitwise identical [B] distortions:
//   pixel   e = fma(db,db, fma(dg,dg, dr*dr))            fp32, round-to-nearest, this order
//   warp    xor-butterfly 16,8,4,2,1 in double           (commutative => all lanes hold the same bits)
//   tile    warps 0..7 added in index order in double    -> partial[state, tile]
//   state   k_distortion_finalize: lane l adds tiles l, l+32, ... in order, then the same butterfly
#pragma once
#include <cuda_runtime.h>

namespace gsr {

__device__ __forceinline__ float pixel_sq_err(float o0, float o1, float o2, float r0, float r1, float r2) {
  const float d0 = __fsub_rn(o0, r0), d1 = __fsub_rn(o1, r1), d2 = __fsub_rn(o2, r2);
  return __fmaf_rn(d2, d2, __fmaf_rn(d1, d1, __fmul_rn(d0, d0)));
}

__device__ __forceinline__ double warp_sum_butterfly(double v) {
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) v += __shfl_xor_sync(0xffffffffu, v, off);
  return v;
}

// The same butterfly for S values per lane at once (S a power of two <= 32), at a fraction of the shuffles:
// at the first steps the two lanes of a pair split the slots between them (each sends the half it gives up
// and adds what it receives to the half it keeps), then the usual butterfly runs on the one slot left.
// For every slot the additions are the pairings lane ^ 16, ^ 8, ... of warp_sum_butterfly, and a + b == b + a
// bitwise, so each slot's total has exactly the bits the plain butterfly gives.  On return every lane holds
// the total of slot `slot`; lanes with (lane & (32 / S - 1)) == 0 are one representative per slot.
template <int S>
__device__ __forceinline__ double warp_sum_slots(double (&v)[S], int lane, int& slot) {
  int off = 16;
  slot = 0;
#pragma unroll
  for (int n = S; n > 1; n >>= 1) {
    const int half = n >> 1;
    const bool upper = (lane & off) != 0;
#pragma unroll
    for (int j = 0; j < half; ++j) {
      const double send = upper ? v[j] : v[j + half];
      const double keep = upper ? v[j + half] : v[j];
      v[j] = keep + __shfl_xor_sync(0xffffffffu, send, off);
    }
    slot = 2 * slot + (upper ? 1 : 0);
    off >>= 1;
  }
  for (; off > 0; off >>= 1) v[0] += __shfl_xor_sync(0xffffffffu, v[0], off);
  return v[0];
}

}  // namespace gsr
