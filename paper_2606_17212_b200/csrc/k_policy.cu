// k_policy.cu — scheduling frontier and partial-state atlas:
//   wire bytes of a completion group       PAPER.md:72   (reading F1)
//   greedy dependency-closed policy orders PAPER.md:96, 130 (reading F2)
//   prefix states at matched byte budgets  PAPER.md:96   (reading F3)
//   wire cost of a sampled state, best sampled state per budget ("empirical oracle") PAPER.md:130 (reading F4)
// All of it is integer / comparison work on [4C]- and [B]-sized arrays: latency-bound helpers around the
// renderer (which produces the PSNR these consume).  Every result is bit-exact and order-independent:
// argmin / argmax ties are broken by the written key, never by thread scheduling.
#include "gsr_internal.h"

namespace gsr {

constexpr int kPolThreads = 256;

// ---- F1: wire = raw + ceil(raw / 1200) * (48 + 4 l), l = g & 3
__global__ void k_wire_bytes(const long long* __restrict__ raw, int n, long long* __restrict__ wire) {
  const int g = blockIdx.x * blockDim.x + threadIdx.x;
  if (g >= n) return;
  const long long r = raw[g];
  const long long chunks = (r + 1199) / 1200;
  wire[g] = r + chunks * (48 + 4 * (long long)(g & 3));
}

// order-preserving integer image of a double (finite values; the caller removes -0 first)
__device__ __forceinline__ unsigned long long ordered_key_f64(double v) {
  unsigned long long u = (unsigned long long)__double_as_longlong(v);
  return (u & 0x8000000000000000ull) ? ~u : (u | 0x8000000000000000ull);
}

struct PolKey {
  unsigned long long primary;  // smaller is better
  unsigned int lc;             // l * C + c : the (l, c) tie-break
  int g;                       // -1: no candidate
};

__device__ __forceinline__ bool better(const PolKey& a, const PolKey& b) {
  if (b.g < 0) return a.g >= 0;
  if (a.g < 0) return false;
  if (a.primary != b.primary) return a.primary < b.primary;
  return a.lc < b.lc;
}

// ---- F2: one CTA builds the whole order (4C sequential picks, each an argmin over <= C eligible groups)
__global__ void __launch_bounds__(kPolThreads) k_frontier_order(const double* __restrict__ score,
                                                                const long long* __restrict__ wire, int C,
                                                                int policy, int* __restrict__ order,
                                                                long long* __restrict__ cum) {
  extern __shared__ unsigned char s_next[];  // [C] next undelivered level of each cluster (4 = exhausted)
  __shared__ PolKey s_best[kPolThreads / 32];
  const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
  for (int c = tid; c < C; c += kPolThreads) s_next[c] = 0;
  __syncthreads();
  long long acc = 0;
  for (int step = 0; step < 4 * C; ++step) {
    PolKey mine{0ull, 0u, -1};
    for (int c = tid; c < C; c += kPolThreads) {
      const int l = s_next[c];
      if (l > 3) continue;
      const int g = 4 * c + l;
      PolKey k;
      k.g = g;
      k.lc = (unsigned)l * (unsigned)C + (unsigned)c;
      if (policy == GSR_POLICY_UTILITY) {
        // key -score ascending; "+ 0.0" turns -0 into +0 so that equal scores compare equal as integers
        k.primary = ordered_key_f64(-score[g] + 0.0);
      } else if (policy == GSR_POLICY_NOMINAL) {
        k.primary = 0ull;
      } else {
        k.primary = (unsigned long long)wire[g] ^ 0x8000000000000000ull;  // signed -> ordered unsigned
      }
      if (better(k, mine)) mine = k;
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
      PolKey o;
      o.primary = __shfl_xor_sync(0xffffffffu, mine.primary, off);
      o.lc = __shfl_xor_sync(0xffffffffu, mine.lc, off);
      o.g = __shfl_xor_sync(0xffffffffu, mine.g, off);
      if (better(o, mine)) mine = o;
    }
    if (lane == 0) s_best[w] = mine;
    __syncthreads();
    if (tid == 0) {
      PolKey b = s_best[0];
      for (int k = 1; k < kPolThreads / 32; ++k)
        if (better(s_best[k], b)) b = s_best[k];
      s_next[b.g >> 2] += 1;
      acc += wire[b.g];
      order[step] = b.g;
      if (cum) cum[step] = acc;
    }
    __syncthreads();
  }
}

// ---- F3: thread j walks the order for budget j: longest prefix with cumulative wire bytes <= budget
__global__ void k_frontier_states(const int* __restrict__ order, const long long* __restrict__ wire, int C,
                                  const long long* __restrict__ budgets, int nb, signed char* __restrict__ levels,
                                  long long* __restrict__ used, int* __restrict__ n_groups, int* __restrict__ err) {
  const int j = blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= nb) return;
  signed char* row = levels + (size_t)j * C;
  for (int c = 0; c < C; ++c) row[c] = -1;
  const long long beta = budgets[j];
  long long acc = 0;
  int n = 0;
  for (int k = 0; k < 4 * C; ++k) {
    const int g = order[k];
    if ((unsigned)g >= 4u * (unsigned)C) {  // not a group id: the walk stops here, the caller is told
      if (err) atomicOr(err, kBadOrder);
      break;
    }
    const long long wg = wire[g];
    if (acc + wg > beta) break;
    acc += wg;
    row[g >> 2] += 1;
    ++n;
  }
  if (used) used[j] = acc;
  if (n_groups) n_groups[j] = n;
}

// ---- wire cost of a dependency-closed state: one warp per state, lanes strided over clusters
__global__ void __launch_bounds__(kPolThreads) k_state_bytes(const signed char* __restrict__ levels, int B, int C,
                                                             const long long* __restrict__ wire,
                                                             long long* __restrict__ out) {
  const int b = blockIdx.x * (kPolThreads / 32) + (threadIdx.x >> 5), lane = threadIdx.x & 31;
  if (b >= B) return;
  long long acc = 0;
  for (int c = lane; c < C; c += 32) {
    const int d = levels[(size_t)b * C + c];
    for (int l = 0; l <= d && l < 4; ++l) acc += wire[4 * c + l];
  }
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, off);  // integer: order-free
  if (lane == 0) out[b] = acc;
}

// ---- F4: CTA j finds argmax psnr over states with bytes <= budget j; ties -> lowest index; none -> -1
__global__ void __launch_bounds__(kPolThreads) k_best_under_budget(const float* __restrict__ psnr,
                                                                   const long long* __restrict__ bytes, int B,
                                                                   const long long* __restrict__ budgets,
                                                                   int* __restrict__ best) {
  __shared__ float s_v[kPolThreads / 32];
  __shared__ int s_i[kPolThreads / 32];
  const int j = blockIdx.x, tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
  const long long beta = budgets[j];
  float v = 0.0f;
  int idx = -1;
  for (int b = tid; b < B; b += kPolThreads) {  // ascending b per thread: '>' keeps the lowest index
    if (bytes[b] <= beta) {
      const float p = psnr[b];
      if (idx < 0 || p > v) { v = p; idx = b; }
    }
  }
  auto merge = [](float& v0, int& i0, float v1, int i1) {
    if (i1 >= 0 && (i0 < 0 || v1 > v0 || (v1 == v0 && i1 < i0))) { v0 = v1; i0 = i1; }
  };
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) {
    const float ov = __shfl_xor_sync(0xffffffffu, v, off);
    const int oi = __shfl_xor_sync(0xffffffffu, idx, off);
    merge(v, idx, ov, oi);
  }
  if (lane == 0) { s_v[w] = v; s_i[w] = idx; }
  __syncthreads();
  if (tid == 0) {
    for (int k = 1; k < kPolThreads / 32; ++k) merge(v, idx, s_v[k], s_i[k]);
    best[j] = idx;
  }
}

// ------------------------------------------------------------------------------------------------ launchers
void launch_wire_bytes(const long long* raw, int32_t C, long long* wire, cudaStream_t st) {
  const int n = 4 * C;
  k_wire_bytes<<<(n + 255) / 256, 256, 0, st>>>(raw, n, wire);
  count_launches(1);
}

void launch_frontier_order(const double* score, const long long* wire, int32_t C, int32_t policy, int32_t* order,
                           long long* cum, cudaStream_t st) {
  k_frontier_order<<<1, kPolThreads, (size_t)C, st>>>(score, wire, C, policy, order, cum);
  count_launches(1);
}

void launch_frontier_states(const int32_t* order, const long long* wire, int32_t C, const long long* budgets,
                            int32_t nb, int8_t* levels, long long* used, int32_t* n_groups, cudaStream_t st) {
  if (nb == 0) return;
  k_frontier_states<<<(nb + 63) / 64, 64, 0, st>>>(order, wire, C, budgets, nb, (signed char*)levels, used, n_groups,
                                                   device_error_word());
  count_launches(1);
}

void launch_state_bytes(const int8_t* levels, int32_t B, int32_t C, const long long* wire, long long* out,
                        cudaStream_t st) {
  if (B == 0) return;
  const int per = kPolThreads / 32;
  k_state_bytes<<<(B + per - 1) / per, kPolThreads, 0, st>>>((const signed char*)levels, B, C, wire, out);
  count_launches(1);
}

void launch_best_under_budget(const float* psnr, const long long* bytes, int32_t B, const long long* budgets,
                              int32_t nb, int32_t* best, cudaStream_t st) {
  if (nb == 0) return;
  k_best_under_budget<<<nb, kPolThreads, 0, st>>>(psnr, bytes, B, budgets, best);
  count_launches(1);
}

}  // namespace gsr
