// k_utility.cu — stage a5b: counterfactual utility, Eq. (3) per pair and Eq. (4) per group
// (DESIGN.md §3.7, §6).
//
//   delta_mse[p] = MSE(m) - MSE(m u g)          Eq. (3) with D = MSE
//   delta_db[p]  = PSNR(m u g) - PSNR(m)        Eq. (3) with D = -PSNR  (unit of the 1e-3 dB tolerance)
//   per group: mean, Q_0.1 (linear interpolation at 0.1 (n-1) of the sorted samples), population std,
//              risk-adjusted utility ((1-a) mean + a Q_0.1) / (1 + b std), a = 0.25, b = 0.05.
//
// One CTA per group.  Members are found by scanning the pair list (group sizes are ~10^2, pair lists
// ~10^3-10^4).  Sums use a fixed order (thread-strided partials, then a fixed shared-memory tree), so
// results are deterministic.  The two order statistics around position 0.1 (n-1) are found by an
// exact radix select on the order-preserving integer image of the doubles — no sort, any group size.
#include "gsr_internal.h"

namespace gsr {

__device__ __forceinline__ unsigned long long ordered_key(double v) {
  unsigned long long u = (unsigned long long)__double_as_longlong(v);
  return (u & 0x8000000000000000ull) ? ~u : (u | 0x8000000000000000ull);
}
__device__ __forceinline__ double from_ordered_key(unsigned long long k) {
  unsigned long long u = (k & 0x8000000000000000ull) ? (k & 0x7FFFFFFFFFFFFFFFull) : ~k;
  return __longlong_as_double((long long)u);
}

constexpr int kUtilThreads = 256;
constexpr int kUtilCap = 2048;  // members cached in shared memory; larger groups re-scan global memory

template <typename T>
__device__ __forceinline__ T block_sum(T v, T* sm) {
  sm[threadIdx.x] = v;
  __syncthreads();
  for (int k = kUtilThreads / 2; k > 0; k >>= 1) {
    if (threadIdx.x < k) sm[threadIdx.x] += sm[threadIdx.x + k];
    __syncthreads();
  }
  T r = sm[0];
  __syncthreads();
  return r;
}

struct PairView {
  const double* mse;
  const float* psnr;
  const int32_t *iwo, *iw, *gid;
  int n_pairs;
  int B;     // states behind mse / psnr; < 0: unknown (only negative indices can then be refused)
  int* err;  // device error word (gsr_index_status) or nullptr
};

// both state indices of pair p usable?
__device__ __forceinline__ bool pair_ok(const PairView& pv, int p) {
  const int a = pv.iwo[p], b = pv.iw[p];
  return a >= 0 && b >= 0 && (pv.B < 0 || (a < pv.B && b < pv.B));
}

__device__ __forceinline__ double pair_delta(const PairView& pv, int p, int metric) {
  return metric == 0 ? pv.mse[pv.iwo[p]] - pv.mse[pv.iw[p]]
                     : (double)pv.psnr[pv.iw[p]] - (double)pv.psnr[pv.iwo[p]];
}

// k-th smallest (0-based) of the group's deltas: MSB-first radix select on ordered keys.
__device__ double select_kth(const PairView& pv, int g, int metric, int n_g, const double* cache, int k,
                             unsigned long long* sm_cnt) {
  unsigned long long ans = 0ull;
  for (int bit = 63; bit >= 0; --bit) {
    const unsigned long long cand = ans | (1ull << bit);
    unsigned long long c = 0;
    if (cache) {
      for (int i = threadIdx.x; i < n_g; i += kUtilThreads) c += ordered_key(cache[i]) < cand;
    } else {
      for (int p = threadIdx.x; p < pv.n_pairs; p += kUtilThreads)
        if (pv.gid[p] == g && pair_ok(pv, p)) c += ordered_key(pair_delta(pv, p, metric)) < cand;
    }
    c = block_sum<unsigned long long>(c, sm_cnt);
    if (c <= (unsigned long long)k) ans = cand;  // at most k keys below cand => the k-th key is >= cand
  }
  return from_ordered_key(ans);
}

__global__ void __launch_bounds__(kUtilThreads) k_pair_delta(PairView pv, double* __restrict__ dmse,
                                                             double* __restrict__ ddb) {
  int p = blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= pv.n_pairs) return;
  if (!pair_ok(pv, p)) {  // refused pair: zero difference, the caller is told
    if (pv.err) atomicOr(pv.err, kBadPairIndex);
    if (dmse) dmse[p] = 0.0;
    if (ddb) ddb[p] = 0.0;
    return;
  }
  if (dmse) dmse[p] = pair_delta(pv, p, 0);
  if (ddb) ddb[p] = pair_delta(pv, p, 1);
}

__global__ void __launch_bounds__(kUtilThreads) k_group_utility(PairView pv, int G, gsr_utility* __restrict__ out) {
  __shared__ double sm_d[kUtilThreads];
  __shared__ unsigned long long sm_c[kUtilThreads];
  __shared__ double cache[kUtilCap];
  __shared__ uint32_t wcnt[8];
  __shared__ uint32_t run_s;
  const int g = blockIdx.x;
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  double res[2][4];
  int n_g = 0;
  if (pv.err && g == 0) {  // one CTA reports group ids no group owns and pairs with unusable state indices
    bool bad_g = false, bad_p = false;
    for (int p = threadIdx.x; p < pv.n_pairs; p += kUtilThreads) {
      const bool in = (unsigned)pv.gid[p] < (unsigned)G;
      bad_g |= !in;
      bad_p |= in && !pair_ok(pv, p);
    }
    if (bad_g) atomicOr(pv.err, kBadGroupId);
    if (bad_p) atomicOr(pv.err, kBadPairIndex);
  }
  for (int metric = 0; metric < 2; ++metric) {
    // ordered compaction of the group's deltas (pair order) into the cache; count members
    if (threadIdx.x == 0) run_s = 0;
    __syncthreads();
    for (int base = 0; base < pv.n_pairs; base += kUtilThreads) {
      const int p = base + threadIdx.x;
      const bool mem = p < pv.n_pairs && pv.gid[p] == g && pair_ok(pv, p);  // a refused pair belongs to no group
      const uint32_t bal = __ballot_sync(0xffffffffu, mem);
      if (lane == 0) wcnt[w] = __popc(bal);
      __syncthreads();
      uint32_t woff = 0, tot = 0;
      for (int q = 0; q < 8; ++q) {
        if (q < w) woff += wcnt[q];
        tot += wcnt[q];
      }
      const uint32_t pos = run_s + woff + __popc(bal & ((1u << lane) - 1u));
      if (mem && pos < kUtilCap) cache[pos] = pair_delta(pv, p, metric);
      __syncthreads();
      if (threadIdx.x == 0) run_s += tot;
      __syncthreads();
    }
    n_g = (int)run_s;
    const bool cached = n_g <= kUtilCap;
    if (n_g == 0) {
      res[metric][0] = res[metric][1] = res[metric][2] = res[metric][3] = 0.0;
      continue;
    }
    // mean
    double s = 0.0;
    if (cached) {
      for (int i = threadIdx.x; i < n_g; i += kUtilThreads) s += cache[i];
    } else {
      for (int p = threadIdx.x; p < pv.n_pairs; p += kUtilThreads)
        if (pv.gid[p] == g && pair_ok(pv, p)) s += pair_delta(pv, p, metric);
    }
    const double mean = block_sum<double>(s, sm_d) / (double)n_g;
    // population variance
    s = 0.0;
    if (cached) {
      for (int i = threadIdx.x; i < n_g; i += kUtilThreads) { const double d = cache[i] - mean; s += d * d; }
    } else {
      for (int p = threadIdx.x; p < pv.n_pairs; p += kUtilThreads)
        if (pv.gid[p] == g && pair_ok(pv, p)) { const double d = pair_delta(pv, p, metric) - mean; s += d * d; }
    }
    const double sd = sqrt(block_sum<double>(s, sm_d) / (double)n_g);
    // Q_0.1 by linear interpolation at position 0.1 (n-1)
    const double posq = 0.1 * (double)(n_g - 1);
    const int lo = (int)floor(posq);
    const int hi = lo + 1 < n_g ? lo + 1 : n_g - 1;
    const double fr = posq - (double)lo;
    double vlo, vhi;
    if (cached) {
      // rank by counting (ties broken by position: ranks are a permutation) — one pass, no sort
      __shared__ double s_sel[2];
      for (int i = threadIdx.x; i < n_g; i += kUtilThreads) {
        const double v = cache[i];
        int r = 0;
        for (int j = 0; j < n_g; ++j) {
          const double c = cache[j];
          r += (c < v) || (c == v && j < i);
        }
        if (r == lo) s_sel[0] = v;
        if (r == hi) s_sel[1] = v;
      }
      __syncthreads();
      vlo = s_sel[0];
      vhi = s_sel[1];
      __syncthreads();
    } else {
      vlo = select_kth(pv, g, metric, n_g, nullptr, lo, sm_c);
      vhi = hi == lo ? vlo : select_kth(pv, g, metric, n_g, nullptr, hi, sm_c);
    }
    const double q10 = vlo + fr * (vhi - vlo);
    const double alpha = 0.25, beta = 0.05;
    res[metric][0] = mean;
    res[metric][1] = q10;
    res[metric][2] = sd;
    res[metric][3] = ((1.0 - alpha) * mean + alpha * q10) / (1.0 + beta * sd);
    __syncthreads();
  }
  if (threadIdx.x == 0) {
    gsr_utility u;
    u.mean_mse = res[0][0]; u.q10_mse = res[0][1]; u.std_mse = res[0][2]; u.risk_mse = res[0][3];
    u.mean_db = res[1][0]; u.q10_db = res[1][1]; u.std_db = res[1][2]; u.risk_db = res[1][3];
    u.count = (double)n_g;
    out[g] = u;
  }
}

void launch_group_utility(const double* mse, const float* psnr, int32_t B, const int32_t* iwo, const int32_t* iw,
                          const int32_t* gid, int32_t n_pairs, int32_t G, gsr_utility* out, double* dmse,
                          double* ddb, cudaStream_t st) {
  PairView pv{mse, psnr, iwo, iw, gid, n_pairs, B, device_error_word()};
  if (n_pairs > 0 && (dmse || ddb))
  {
    k_pair_delta<<<(n_pairs + kUtilThreads - 1) / kUtilThreads, kUtilThreads, 0, st>>>(pv, dmse, ddb);
    count_launches(1);
  }
  if (G > 0) {
    k_group_utility<<<G, kUtilThreads, 0, st>>>(pv, G, out);
    count_launches(1);
  }
}

}  // namespace gsr
