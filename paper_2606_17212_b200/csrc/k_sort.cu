// k_sort.cu — stage a3 of the hot path: tile binning and the key sort.
//
//   K2a  exclusive scan of the per-record tile counts (warp-shuffle segmented scan, 3 phases)
//   K2b  key emission: (tile << 32 | depth bits) with the record id as payload, written at
//        scan offsets — i.e. in ascending record order, no atomics, so the emission is deterministic
//   K3   stable LSD radix sort, 8-bit digits over the 32 + ceil(log2 tiles) significant key bits;
//        ties in (tile, depth) keep emission order = ascending record id = ascending
//        (Gaussian index, variant), which is exactly the (tile, depth, index) order of the spec
//   K3b  per-tile [start, end) ranges
//
// The state field of the spec's (state, tile, depth, index) key is factored out: the sorted list
// of state b is the restriction of this per-frame superset list to the records present in b
// (DESIGN.md §4.2).  k_filter_keys materialises it for the bit-exact parity check and
// k_state_counts gives its length I_b for every state of the batch.
//
// All sizes that depend on the data (number of keys) stay on the device: grids are sized for the
// key capacity and read the actual count from the workspace header, so the whole path is
// asynchronous on the caller's stream.
#include "gsr_internal.h"

namespace gsr {

// ------------------------------------------------------------------------------------------------
// K2a: exclusive scan over n uint32 (n <= 2^31), block = 256 threads x 8 items
constexpr int kScanThreads = 256, kScanItems = 8, kScanTile = kScanThreads * kScanItems;

__device__ __forceinline__ uint32_t warp_incl_scan(uint32_t v) {
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    uint32_t n = __shfl_up_sync(0xffffffffu, v, d);
    if ((threadIdx.x & 31) >= d) v += n;
  }
  return v;
}

// block-wide exclusive scan of one value per thread (256 threads); returns exclusive prefix, total in *total
__device__ __forceinline__ uint32_t block_excl_scan_256(uint32_t v, uint32_t* smem8, uint32_t* total) {
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  uint32_t inc = warp_incl_scan(v);
  if (lane == 31) smem8[w] = inc;
  __syncthreads();
  uint32_t woff = 0, tot = 0;
#pragma unroll
  for (int k = 0; k < 8; ++k) {
    uint32_t s = smem8[k];
    if (k < w) woff += s;
    tot += s;
  }
  __syncthreads();
  *total = tot;
  return woff + inc - v;
}

__global__ void __launch_bounds__(kScanThreads) k_scan_block_sums(const uint32_t* __restrict__ in, int n,
                                                                  uint32_t* __restrict__ blk) {
  __shared__ uint32_t sm[8];
  int base = blockIdx.x * kScanTile + threadIdx.x * kScanItems;
  uint32_t s = 0;
#pragma unroll
  for (int k = 0; k < kScanItems; ++k)
    if (base + k < n) s += in[base + k];
  uint32_t tot;
  block_excl_scan_256(s, sm, &tot);
  if (threadIdx.x == 0) blk[blockIdx.x] = tot;
}

// single CTA: exclusive scan of the block sums in place; total (64-bit) -> header; capacity check
__global__ void __launch_bounds__(kScanThreads) k_scan_top(uint32_t* __restrict__ blk, int nblk, WsHeader* hdr) {
  __shared__ uint32_t sm[8];
  __shared__ unsigned long long carry_s;
  if (threadIdx.x == 0) carry_s = 0ull;
  __syncthreads();
  for (int base = 0; base < nblk; base += kScanThreads) {
    int i = base + threadIdx.x;
    uint32_t v = i < nblk ? blk[i] : 0u;
    uint32_t tot;
    uint32_t ex = block_excl_scan_256(v, sm, &tot);
    unsigned long long carry = carry_s;
    if (i < nblk) blk[i] = (uint32_t)(carry + ex);  // meaningful only while the total fits the capacity (< 2^31)
    __syncthreads();
    if (threadIdx.x == 0) carry_s = carry + tot;
    __syncthreads();
  }
  if (threadIdx.x == 0) {
    unsigned long long total = carry_s;
    hdr->total_keys = total;
    if ((long long)total > hdr->key_capacity) {
      atomicMin(&hdr->status, GSR_E_WORKSPACE_TOO_SMALL);
      hdr->n_keys = 0ull;  // render nothing rather than a truncated (wrong) list
    } else {
      hdr->n_keys = total;
    }
  }
}

__global__ void __launch_bounds__(kScanThreads) k_scan_apply(const uint32_t* __restrict__ in, int n,
                                                             const uint32_t* __restrict__ blk,
                                                             uint32_t* __restrict__ out) {
  __shared__ uint32_t sm[8];
  int base = blockIdx.x * kScanTile + threadIdx.x * kScanItems;
  uint32_t v[kScanItems], s = 0;
#pragma unroll
  for (int k = 0; k < kScanItems; ++k) {
    v[k] = (base + k < n) ? in[base + k] : 0u;
    s += v[k];
  }
  uint32_t tot;
  uint32_t ex = block_excl_scan_256(s, sm, &tot) + blk[blockIdx.x];
#pragma unroll
  for (int k = 0; k < kScanItems; ++k) {
    if (base + k < n) out[base + k] = ex;
    ex += v[k];
  }
  if (blockIdx.x == gridDim.x - 1 && threadIdx.x == kScanThreads - 1) out[n] = ex;  // grand total (mod 2^32)
}

// ------------------------------------------------------------------------------------------------
// K2b: one thread per record writes its count keys in (ty, tx) order at [offset, offset + count)
__global__ void __launch_bounds__(256) k_emit_keys(int n_rec, const uint32_t* __restrict__ count,
                                                   const uint32_t* __restrict__ offset,
                                                   const uint2* __restrict__ rect,
                                                   const uint32_t* __restrict__ depth_bits, int TX,
                                                   const WsHeader* __restrict__ hdr,
                                                   unsigned long long* __restrict__ keys,
                                                   uint32_t* __restrict__ vals) {
  int r = blockIdx.x * blockDim.x + threadIdx.x;
  if (r >= n_rec) return;
  if (hdr->n_keys == 0ull) return;
  uint32_t cnt = count[r];
  if (cnt == 0) return;
  uint32_t o = offset[r];
  uint2 rc = rect[r];
  int tx0 = rc.x & 0xFFFF, ty0 = rc.x >> 16, tx1 = rc.y & 0xFFFF, ty1 = rc.y >> 16;
  unsigned long long d = depth_bits[r];
  for (int ty = ty0; ty < ty1; ++ty)
    for (int tx = tx0; tx < tx1; ++tx) {
      keys[o] = ((unsigned long long)(uint32_t)(ty * TX + tx) << 32) | d;
      vals[o] = (uint32_t)r;
      ++o;
    }
}

// ------------------------------------------------------------------------------------------------
// K3: stable LSD radix sort, one 8-bit digit per pass.
//   hist    : per-block digit counts, layout [digit][block]
//   scan    : exclusive scan over that array in (digit, block) order (single CTA)
//   scatter : stable in-block ranking (warp match + per-warp counters), then write
__global__ void __launch_bounds__(kSortThreads) k_radix_hist(const unsigned long long* __restrict__ keys,
                                                            const WsHeader* __restrict__ hdr, int shift,
                                                            uint32_t* __restrict__ hist) {
  const unsigned long long n = hdr->n_keys;
  const unsigned long long base = (unsigned long long)blockIdx.x * kSortTileKeys;
  if (base >= n) return;
  const uint32_t nblk = (uint32_t)((n + kSortTileKeys - 1) / kSortTileKeys);
  __shared__ uint32_t h[256];
  h[threadIdx.x] = 0;
  __syncthreads();
#pragma unroll 4
  for (int k = 0; k < kSortItems; ++k) {
    unsigned long long i = base + (unsigned long long)k * kSortThreads + threadIdx.x;
    if (i < n) atomicAdd(&h[(uint32_t)(keys[i] >> shift) & 0xFFu], 1u);
  }
  __syncthreads();
  hist[(size_t)threadIdx.x * nblk + blockIdx.x] = h[threadIdx.x];
}

// one warp per digit: exclusive prefix of that digit's per-block counts (in place) and the digit total,
// stored behind the table at hist[256 * nblk + digit]; the scatter kernel scans the 256 totals itself
__global__ void __launch_bounds__(256) k_radix_scan(uint32_t* __restrict__ hist, const WsHeader* __restrict__ hdr) {
  const unsigned long long n = hdr->n_keys;
  const uint32_t nblk = (uint32_t)((n + kSortTileKeys - 1) / kSortTileKeys);
  const int lane = threadIdx.x & 31;
  const uint32_t d = blockIdx.x * 8 + (threadIdx.x >> 5);
  uint32_t* row = hist + (size_t)d * nblk;
  uint32_t carry = 0;
  for (uint32_t base = 0; base < nblk; base += 32) {
    const uint32_t b = base + lane;
    const uint32_t v = b < nblk ? row[b] : 0u;
    const uint32_t inc = warp_incl_scan(v);
    if (b < nblk) row[b] = carry + inc - v;
    carry += __shfl_sync(0xffffffffu, inc, 31);
  }
  if (lane == 0) hist[(size_t)256 * nblk + d] = carry;
}

__global__ void __launch_bounds__(kSortThreads) k_radix_scatter(const unsigned long long* __restrict__ keys_in,
                                                               const uint32_t* __restrict__ vals_in,
                                                               unsigned long long* __restrict__ keys_out,
                                                               uint32_t* __restrict__ vals_out,
                                                               const WsHeader* __restrict__ hdr, int shift,
                                                               const uint32_t* __restrict__ hist) {
  const unsigned long long n = hdr->n_keys;
  const unsigned long long base = (unsigned long long)blockIdx.x * kSortTileKeys;
  if (base >= n) return;
  const uint32_t nblk = (uint32_t)((n + kSortTileKeys - 1) / kSortTileKeys);
  __shared__ uint32_t cnt[kSortThreads / 32][256];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  for (int k = threadIdx.x; k < (kSortThreads / 32) * 256; k += kSortThreads) (&cnt[0][0])[k] = 0;
  __syncthreads();
  // warp w owns the contiguous chunk [base + w*512, base + (w+1)*512): stable order = (warp, round, lane)
  unsigned long long key[kSortItems];
  uint32_t val[kSortItems], rank[kSortItems];
  const unsigned long long wbase = base + (unsigned long long)w * (32 * kSortItems);
#pragma unroll
  for (int k = 0; k < kSortItems; ++k) {
    unsigned long long i = wbase + (unsigned long long)k * 32 + lane;
    bool ok = i < n;
    key[k] = ok ? keys_in[i] : ~0ull;
    val[k] = ok ? vals_in[i] : 0u;
  }
#pragma unroll
  for (int k = 0; k < kSortItems; ++k) {
    unsigned long long i = wbase + (unsigned long long)k * 32 + lane;
    bool ok = i < n;
    uint32_t d = ok ? ((uint32_t)(key[k] >> shift) & 0xFFu) : 256u;  // 256 = "no key", never counted
    uint32_t peers = __match_any_sync(0xffffffffu, d);
    uint32_t lt = peers & ((1u << lane) - 1u);
    uint32_t b = 0;
    if (ok) b = cnt[w][d];
    __syncwarp();
    if (ok && lt == 0) cnt[w][d] = b + __popc(peers);
    __syncwarp();
    rank[k] = b + __popc(lt);
  }
  __syncthreads();
  {  // per digit: exclusive prefix over warps + the block's global base
    //   base(d) = sum of the totals of digits < d  +  this digit's count in earlier blocks
    const int d = threadIdx.x;
    __shared__ uint32_t s_w8[8];
    const uint32_t tot = hist[(size_t)256 * nblk + d];
    const uint32_t inc = warp_incl_scan(tot);
    if (lane == 31) s_w8[w] = inc;
    __syncthreads();
    uint32_t dbase = inc - tot;
    for (int ww = 0; ww < w; ++ww) dbase += s_w8[ww];
    uint32_t acc = hist[(size_t)d * nblk + blockIdx.x] + dbase;
#pragma unroll
    for (int ww = 0; ww < kSortThreads / 32; ++ww) {
      uint32_t c = cnt[ww][d];
      cnt[ww][d] = acc;
      acc += c;
    }
  }
  __syncthreads();
#pragma unroll
  for (int k = 0; k < kSortItems; ++k) {
    unsigned long long i = wbase + (unsigned long long)k * 32 + lane;
    if (i < n) {
      uint32_t d = (uint32_t)(key[k] >> shift) & 0xFFu;
      uint32_t pos = cnt[w][d] + rank[k];
      keys_out[pos] = key[k];
      vals_out[pos] = val[k];
    }
  }
}

// K3b: tile ranges from the sorted keys
__global__ void __launch_bounds__(256) k_tile_ranges(const unsigned long long* __restrict__ keys,
                                                     const WsHeader* __restrict__ hdr, uint2* __restrict__ range) {
  const unsigned long long n = hdr->n_keys;
  for (unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; i < n;
       i += (unsigned long long)gridDim.x * blockDim.x) {
    uint32_t t = (uint32_t)(keys[i] >> 32);
    if (i == 0 || (uint32_t)(keys[i - 1] >> 32) != t) range[t].x = (uint32_t)i;
    if (i + 1 == n || (uint32_t)(keys[i + 1] >> 32) != t) range[t].y = (uint32_t)(i + 1);
  }
}

void launch_bin_and_sort(const DeviceScene& sc, const FrameParams& fp, Workspace& ws, long long cap,
                         cudaStream_t st) {
  const int n_rec = sc.V * sc.N;
  const int tiles = fp.TX * fp.TY;
  cudaMemsetAsync(ws.tile_range, 0, sizeof(uint2) * (size_t)tiles, st);
  if (n_rec == 0) return;
  const int nblk = (n_rec + kScanTile - 1) / kScanTile;
  k_scan_block_sums<<<nblk, kScanThreads, 0, st>>>(ws.count, n_rec, ws.scan_blk);
  k_scan_top<<<1, kScanThreads, 0, st>>>(ws.scan_blk, nblk, ws.hdr);
  k_scan_apply<<<nblk, kScanThreads, 0, st>>>(ws.count, n_rec, ws.scan_blk, ws.offset);
  k_emit_keys<<<(n_rec + 255) / 256, 256, 0, st>>>(n_rec, ws.count, ws.offset, ws.rect, ws.depth_bits, fp.TX,
                                                   ws.hdr, ws.keys[0], ws.vals[0]);
  // significant bits: 32 depth bits + tile bits, rounded up to whole 8-bit digits
  int tile_bits = 1;
  while ((1 << tile_bits) < tiles) ++tile_bits;
  int passes = (32 + tile_bits + 7) / 8;
  if (passes & 1) ++passes;  // an even number of passes leaves the result in buffer 0
  const unsigned sort_blocks = (unsigned)((cap + kSortTileKeys - 1) / kSortTileKeys);
  for (int p = 0; p < passes; ++p) {
    const int in = p & 1, out = in ^ 1, shift = 8 * p;
    k_radix_hist<<<sort_blocks, kSortThreads, 0, st>>>(ws.keys[in], ws.hdr, shift, ws.hist);
    k_radix_scan<<<32, 256, 0, st>>>(ws.hist, ws.hdr);
    k_radix_scatter<<<sort_blocks, kSortThreads, 0, st>>>(ws.keys[in], ws.vals[in], ws.keys[out], ws.vals[out],
                                                          ws.hdr, shift, ws.hist);
  }
  k_tile_ranges<<<148 * 8, 256, 0, st>>>(ws.keys[0], ws.hdr, ws.tile_range);
  count_launches(4 + 3 * passes + 1);
}

// ------------------------------------------------------------------------------------------------
// presence of record r (class cls of cluster c) in a state whose cluster depth is d:
//   cls 0 (variant A, level-0 Gaussian): d == 0 ; cls 1+l (variant B, level l): d >= max(1, l)
__device__ __forceinline__ bool record_present(uint32_t cls, int d) {
  if (cls >= 16) return d == (int)cls - 16;  // 4-variant scenes (reading I1): variant v lives in depth v only
  return cls == 0 ? (d == 0) : (d >= 1 && d >= (int)cls - 1);
}

// I_b for every state: sum over records of count * present.  One CTA per state, fixed tree (integers).
__global__ void __launch_bounds__(256) k_state_counts(int n_rec, const uint32_t* __restrict__ count,
                                                      const float4* __restrict__ r1,
                                                      const int8_t* __restrict__ depth, int C,
                                                      long long* __restrict__ out) {
  const int b = blockIdx.x;
  long long s = 0;
  for (int r = threadIdx.x; r < n_rec; r += blockDim.x) {
    uint32_t cnt = count[r];
    if (cnt == 0) continue;
    uint32_t meta = __float_as_uint(r1[r].w);
    int d = depth[(size_t)b * C + (meta & 0xFFFFu)];
    if (record_present(meta >> 16, d)) s += cnt;
  }
  __shared__ long long sm[256];
  sm[threadIdx.x] = s;
  __syncthreads();
  for (int k = 128; k > 0; k >>= 1) {
    if (threadIdx.x < k) sm[threadIdx.x] += sm[threadIdx.x + k];
    __syncthreads();
  }
  if (threadIdx.x == 0) out[b] = sm[0];
}

void launch_state_counts(const DeviceScene& sc, Workspace& ws, int32_t B, cudaStream_t st) {
  if (B == 0) return;
  k_state_counts<<<B, 256, 0, st>>>(sc.V * sc.N, ws.count, ws.r1, ws.depth, sc.C, ws.state_counts);
  count_launches(1);
}

// Debug: the literal (tile, depth bits, Gaussian) list of state b = ordered filter of the superset list.
// Single CTA, ordered compaction by ballot + running offset.
__global__ void __launch_bounds__(256) k_filter_keys(const unsigned long long* __restrict__ keys,
                                                     const uint32_t* __restrict__ vals,
                                                     const WsHeader* __restrict__ hdr,
                                                     const float4* __restrict__ r1,
                                                     const int8_t* __restrict__ depth, int C, int V, int b,
                                                     uint32_t* __restrict__ tile, uint32_t* __restrict__ dbits,
                                                     int32_t* __restrict__ gi, unsigned long long* n_out,
                                                     long long cap) {
  const unsigned long long n = hdr->n_keys;
  __shared__ uint32_t wcnt[8];
  __shared__ unsigned long long run_s;
  if (threadIdx.x == 0) run_s = 0;
  __syncthreads();
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  for (unsigned long long base = 0; base < n; base += 256) {
    unsigned long long i = base + threadIdx.x;
    bool keep = false;
    unsigned long long k = 0;
    uint32_t rid = 0;
    if (i < n) {
      k = keys[i];
      rid = vals[i];
      uint32_t meta = __float_as_uint(r1[rid].w);
      int d = depth[(size_t)b * C + (meta & 0xFFFFu)];
      keep = record_present(meta >> 16, d);
    }
    uint32_t bal = __ballot_sync(0xffffffffu, keep);
    if (lane == 0) wcnt[w] = __popc(bal);
    __syncthreads();
    uint32_t woff = 0, tot = 0;
    for (int q = 0; q < 8; ++q) {
      if (q < w) woff += wcnt[q];
      tot += wcnt[q];
    }
    unsigned long long pos = run_s + woff + __popc(bal & ((1u << lane) - 1u));
    if (keep && (long long)pos < cap) {
      tile[pos] = (uint32_t)(k >> 32);
      dbits[pos] = (uint32_t)k;
      gi[pos] = (int32_t)(rid / (uint32_t)V);
    }
    __syncthreads();
    if (threadIdx.x == 0) run_s += tot;
    __syncthreads();
  }
  if (threadIdx.x == 0) *n_out = run_s;
}

void launch_filter_keys(const DeviceScene& sc, Workspace& ws, int32_t b, uint32_t* tile, uint32_t* dbits,
                        int32_t* gi, unsigned long long* n_out, long long cap, cudaStream_t st) {
  k_filter_keys<<<1, 256, 0, st>>>(ws.keys[0], ws.vals[0], ws.hdr, ws.r1, ws.depth, sc.C, sc.V, b, tile, dbits, gi,
                                   n_out, cap);
}

}  // namespace gsr
