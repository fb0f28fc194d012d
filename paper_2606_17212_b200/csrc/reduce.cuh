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

}  // namespace gsr
