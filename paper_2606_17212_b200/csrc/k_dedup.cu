// k_dedup.cu — tile-level state dedup.
//
// The pixels of a tile in state b depend on b only through the delivered depths of the clusters that
// have records in that tile — and, per such cluster, only through which of the tile's record classes
// the depth makes present (and whether the SH residual applies).  Two states that agree on that
// restricted signature produce bitwise identical tile pixels, so the tile is composited once per
// distinct signature and the result is written to every state that shares it.  (Pairs m, m u g of the
// utility workload differ in ONE cluster: they share every tile that cluster does not touch.)
//
// One CTA per tile:
//   1. class presence bits per cluster from the tile's record list
//   2. per present cluster, the canonical code (0..4) of each depth -1..3 (equal code <=> same signature);
//      the present clusters are ordered by DESCENDING record count in the tile, so that the sort below makes
//      consecutive classes agree on the clusters that carry most of the tile's records: a compositing CTA
//      takes S consecutive classes, and a record it stages is then present in (nearly) all or none of them
//   3. per state a 64-bit key: the packed codes if they fit (3 bits x <= 21 clusters), else the packed codes
//      of the 13 heaviest clusters followed by a 24-bit hash of all of them
//   4. in-CTA bitonic sort of (key, state); a state starts a new class unless its restricted code vector
//      EQUALS its predecessor's (verified exactly, so a hash collision can only cost dedup, never
//      correctness)
//   5. outputs: order[tile][i] = states in sorted order, upos[tile][u] = start of class u, n_unique[tile]
#include "gsr_internal.h"

namespace gsr {

constexpr int kDedupThreads = 256;

__device__ __forceinline__ uint32_t class_sig(uint32_t bits, int d) {
  // bits: 1 = variant-A records (present iff d == 0), 2 = variant-B level 0/1 (d >= 1),
  //       4 = variant-B level 2 (d >= 2), 8 = variant-B level 3 (d >= 3); SH residual iff d == 3 (any B)
  //       16 << v = records of variant v of a 4-variant scene (present iff d == v)
  uint32_t s = 0;
  if ((bits & 1u) && d == 0) s |= 1u;
  if ((bits & 2u) && d >= 1) s |= 2u;
  if ((bits & 4u) && d >= 2) s |= 4u;
  if ((bits & 8u) && d >= 3) s |= 8u;
  if (s >= 2u && d == 3) s |= 256u;  // a present B record takes the residual colour
  if (d >= 0 && ((bits >> (4 + d)) & 1u)) s |= 16u << d;
  return s;
}

__global__ void __launch_bounds__(kDedupThreads) k_tile_dedup(const uint2* __restrict__ tile_range,
                                                              const uint32_t* __restrict__ vals,
                                                              const float4* __restrict__ r1,
                                                              const int8_t* __restrict__ depth, int B, int C,
                                                              int Bp, uint32_t* __restrict__ order,
                                                              uint32_t* __restrict__ upos,
                                                              uint32_t* __restrict__ n_unique) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  // layout: keys u64[Bp] | idx u32[Bp] | head u32[Bp] | cbits u32[ceil(C/4)] | ccnt u32[C] | klist0 u16[C] |
  //         klist u16[C] | codes0 u8[5*C] | codes u8[5*C]
  unsigned long long* keys = (unsigned long long*)smem_raw;
  uint32_t* idx = (uint32_t*)(keys + Bp);
  uint32_t* head = idx + Bp;
  uint32_t* cbits = head + Bp;
  const int cwords = (C + 3) / 4;
  uint32_t* ccnt = cbits + cwords;
  uint16_t* klist0 = (uint16_t*)(ccnt + C);
  uint16_t* klist = klist0 + ((C + 1) & ~1);
  uint8_t* codes0 = (uint8_t*)(klist + ((C + 1) & ~1));
  uint8_t* codes = codes0 + 5 * (size_t)C;
  __shared__ uint32_t s_cnt[8];
  __shared__ uint32_t s_run;

  const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
  const int tile = blockIdx.x;
  const uint2 rg = tile_range[tile];

  // 1. class presence bits
  for (int k = tid; k < cwords; k += kDedupThreads) cbits[k] = 0;
  for (int k = tid; k < C; k += kDedupThreads) ccnt[k] = 0;
  __syncthreads();
  for (uint32_t i = rg.x + tid; i < rg.y; i += kDedupThreads) {
    const uint32_t rid = vals[i];  // render list: sub-tile-culled records are already gone (tile_render_lists in k_sort.cu)
    const uint32_t meta = __float_as_uint(r1[rid].w);
    const uint32_t c = meta & 0xFFFFu, cls = meta >> 16;
    const uint32_t bit = cls >= 16 ? (16u << (cls - 16)) : (cls == 0 ? 1u : (cls <= 2 ? 2u : (cls == 3 ? 4u : 8u)));
    atomicOr(&cbits[c >> 2], bit << (8 * (c & 3)));
    atomicAdd(&ccnt[c], 1u);
  }
  if (tid == 0) s_run = 0;
  __syncthreads();
  // 2. ordered list of present clusters + their depth codes
  for (int base = 0; base < C; base += kDedupThreads) {
    const int c = base + tid;
    const uint32_t bits = c < C ? (cbits[c >> 2] >> (8 * (c & 3))) & 0xFFu : 0u;
    const bool present = bits != 0;
    const uint32_t bal = __ballot_sync(0xffffffffu, present);
    if (lane == 0) s_cnt[w] = __popc(bal);
    __syncthreads();
    uint32_t woff = 0, tot = 0;
    for (int q = 0; q < 8; ++q) {
      if (q < w) woff += s_cnt[q];
      tot += s_cnt[q];
    }
    if (present) {
      const uint32_t pos = s_run + woff + __popc(bal & ((1u << lane) - 1u));
      klist0[pos] = (uint16_t)c;
      uint32_t sig[5];
      for (int d = -1; d <= 3; ++d) sig[d + 1] = class_sig(bits, d);
      for (int d = 0; d < 5; ++d) {
        int code = d;
        for (int e = d - 1; e >= 0; --e)
          if (sig[e] == sig[d]) code = e;
        codes0[5 * pos + d] = (uint8_t)code;
      }
    }
    __syncthreads();
    if (tid == 0) s_run += tot;
    __syncthreads();
  }
  const int k = (int)s_run;
  const bool packed = 3 * k <= 63;
  // order the present clusters by descending record count (rank sort; index order beyond 512 clusters)
  for (int j = tid; j < k; j += kDedupThreads) {
    int rank = j;
    if (k <= 512) {
      const uint32_t mine = ccnt[klist0[j]];
      rank = 0;
      for (int i = 0; i < k; ++i) {
        const uint32_t other = ccnt[klist0[i]];
        rank += (other > mine) || (other == mine && i < j);
      }
    }
    klist[rank] = klist0[j];
    for (int d = 0; d < 5; ++d) codes[5 * rank + d] = codes0[5 * j + d];
  }
  __syncthreads();

  // 3. keys
  for (int b = tid; b < Bp; b += kDedupThreads) {
    unsigned long long key = ~0ull;
    if (b < B) {
      key = 0ull;
      unsigned long long h = 0ull;
      const int8_t* row = depth + (size_t)b * C;
      for (int j = 0; j < k; ++j) {
        const unsigned long long code = codes[5 * j + row[klist[j]] + 1];
        if (packed || j < 13) key = (key << 3) | code;
        if (!packed) h = (h ^ code) * 0x9E3779B97F4A7C15ull + 0x632BE59BD9B4E019ull;
      }
      if (!packed) key = (key << 24) | (h >> 40);  // 39 + 24 bits: real keys stay below the padding key
    }
    keys[b] = key;
    idx[b] = b < B ? (uint32_t)b : 0xFFFFFFFFu;
  }
  __syncthreads();
  // 4. bitonic sort by (key, idx)
  for (int size = 2; size <= Bp; size <<= 1) {
    for (int stride = size >> 1; stride > 0; stride >>= 1) {
      for (int t = tid; t < (Bp >> 1); t += kDedupThreads) {
        const int lo = 2 * t - (t & (stride - 1));
        const int hi = lo + stride;
        const bool asc = (lo & size) == 0;
        const unsigned long long ka = keys[lo], kb = keys[hi];
        const uint32_t ia = idx[lo], ib = idx[hi];
        const bool gt = ka > kb || (ka == kb && ia > ib);
        if (gt == asc) {
          keys[lo] = kb; keys[hi] = ka;
          idx[lo] = ib; idx[hi] = ia;
        }
      }
      __syncthreads();
    }
  }
  // class heads (exact verification against the predecessor)
  for (int i = tid; i < Bp; i += kDedupThreads) {
    uint32_t h = 0;
    if (i < B) {
      if (i == 0 || keys[i] != keys[i - 1]) {
        h = 1;
      } else if (!packed) {
        const int8_t* ra = depth + (size_t)idx[i] * C;
        const int8_t* rb = depth + (size_t)idx[i - 1] * C;
        for (int j = 0; j < k; ++j) {
          const int c = klist[j];
          if (codes[5 * j + ra[c] + 1] != codes[5 * j + rb[c] + 1]) { h = 1; break; }
        }
      }
    }
    head[i] = h;
  }
  if (tid == 0) s_run = 0;
  __syncthreads();
  // 5. ordered compaction of heads -> upos, and the sorted order
  for (int base = 0; base < B; base += kDedupThreads) {
    const int i = base + tid;
    const bool is_head = i < B && head[i] != 0;
    const uint32_t bal = __ballot_sync(0xffffffffu, is_head);
    if (lane == 0) s_cnt[w] = __popc(bal);
    __syncthreads();
    uint32_t woff = 0, tot = 0;
    for (int q = 0; q < 8; ++q) {
      if (q < w) woff += s_cnt[q];
      tot += s_cnt[q];
    }
    if (i < B) order[(size_t)tile * B + i] = idx[i];
    if (is_head) upos[(size_t)tile * B + s_run + woff + __popc(bal & ((1u << lane) - 1u))] = (uint32_t)i;
    __syncthreads();
    if (tid == 0) s_run += tot;
    __syncthreads();
  }
  if (tid == 0) n_unique[tile] = s_run;
}

size_t dedup_smem_bytes(int B, int C, int* Bp_out) {
  int Bp = 2;
  while (Bp < B) Bp <<= 1;
  *Bp_out = Bp;
  return (size_t)Bp * 16 + (size_t)((C + 3) / 4) * 4 + (size_t)C * 4 + 2 * (size_t)((C + 1) & ~1) * 2 + (size_t)10 * C + 16;
}

// Returns false (and launches nothing) if the batch is too large for the in-CTA sort.
bool launch_tile_dedup(const DeviceScene& sc, const FrameParams& fp, Workspace& ws, const int8_t* depth_rows,
                       int32_t B, cudaStream_t st) {
  int Bp = 0;
  const size_t smem = dedup_smem_bytes(B, sc.C, &Bp);
  if (B < 2 || smem > 200 * 1024) return false;
  // the opt-in is per device and cheap: made whenever it is needed rather than once per process
  if (smem > 48 * 1024) cudaFuncSetAttribute(k_tile_dedup, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
  k_tile_dedup<<<fp.TX * fp.TY, kDedupThreads, smem, st>>>(ws.render_range, ws.vals[1], ws.r1, depth_rows, B, sc.C, Bp,
                                                          ws.uorder, ws.upos, ws.n_unique);
  count_launches(1);
  return true;
}

}  // namespace gsr
