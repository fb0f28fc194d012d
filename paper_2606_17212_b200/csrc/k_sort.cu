// k_sort.cu — stage a3 of the hot path: tile binning and the key sort.
//
// The spec's order inside a tile is (depth bits, Gaussian index, variant) = (depth bits, record id), and a
// (depth bits, record id) pair is unique: the sorted list of a tile is a function of its SET of keys.  The sort
// therefore does not have to be stable or to see the keys in any particular order, which allows a counting sort
// by tile followed by an independent sort of every tile's segment — 3 kernels per frame (plus the counting inside k_project) instead of a 6-pass
// global radix sort (23 launches, each pass re-reading and re-writing every key):
//   K2a  (in k_project)  per record: one atomic increment per tile of its rectangle        -> tile_cursor
//   K2b  k_tile_offsets  one CTA: exclusive scan over the tiles -> tile_range (start, end), the total number of
//                        keys -> header (capacity check), cursors reset to the segment starts
//   K2c  k_scatter_keys  per record: (depth bits << 32 | record id) into its tiles' segments (atomic cursor: the
//                        order inside a segment is arbitrary at this point)
//   K3   k_tile_sort     one CTA per tile: bitonic sort of the segment by the 64-bit key — in shared memory up to
//                        4096 keys, in place in global memory beyond — then the canonical arrays
//                        keys[0] = (tile << 32 | depth bits), vals[0] = record id that the parity exports read
//
// The state field of the spec's (state, tile, depth, index) key is factored out: the sorted list
// of state b is the restriction of this per-frame superset list to the records present in b
// (DESIGN.md §4.2).  k_filter_keys materialises it for the bit-exact parity check and
// k_state_counts gives its length I_b for every state of the batch.
//
// All sizes that depend on the data (number of keys) stay on the device, so the whole path is asynchronous on
// the caller's stream.
#include "gsr_internal.h"

namespace gsr {

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

// ------------------------------------------------------------------------------------------------
// K2b: one CTA.  tile_range[t] = [start, end) of tile t's segment, cursor[t] = start; total -> header.
__global__ void __launch_bounds__(256) k_tile_offsets(uint32_t* __restrict__ tile_cursor, int tiles,
                                                      uint2* __restrict__ tile_range, WsHeader* hdr) {
  __shared__ uint32_t sm[8];
  __shared__ unsigned long long carry_s;
  if (threadIdx.x == 0) carry_s = 0ull;
  __syncthreads();
  // first the total (64-bit) and the capacity check: beyond the capacity nothing is binned at all
  unsigned long long part = 0;
  for (int i = threadIdx.x; i < tiles; i += 256) part += tile_cursor[i];
  for (int off = 16; off > 0; off >>= 1) part += __shfl_xor_sync(0xffffffffu, part, off);
  __shared__ unsigned long long s_part[8];
  if ((threadIdx.x & 31) == 0) s_part[threadIdx.x >> 5] = part;
  __syncthreads();
  unsigned long long total = 0;
  for (int k = 0; k < 8; ++k) total += s_part[k];
  const bool fits = (long long)total <= hdr->key_capacity;
  if (threadIdx.x == 0) {
    hdr->total_keys = total;
    if (!fits) atomicMin(&hdr->status, GSR_E_WORKSPACE_TOO_SMALL);
    hdr->n_keys = fits ? total : 0ull;  // render nothing rather than a truncated (wrong) list
  }
  for (int base = 0; base < tiles; base += 256) {
    const int i = base + threadIdx.x;
    const uint32_t v = (i < tiles && fits) ? tile_cursor[i] : 0u;
    uint32_t tot;
    const uint32_t ex = block_excl_scan_256(v, sm, &tot);
    const uint32_t start = (uint32_t)carry_s + ex;
    if (i < tiles) {
      tile_range[i] = make_uint2(start, start + v);
      tile_cursor[i] = start;
    }
    __syncthreads();
    if (threadIdx.x == 0) carry_s += tot;
    __syncthreads();
  }
}

// K2c: every record writes (depth bits << 32 | record id) into the segment of each tile of its rectangle
__global__ void __launch_bounds__(256) k_scatter_keys(int n_rec, const uint32_t* __restrict__ count,
                                                      const uint2* __restrict__ rect,
                                                      const uint32_t* __restrict__ depth_bits, int TX,
                                                      const WsHeader* __restrict__ hdr,
                                                      uint32_t* __restrict__ tile_cursor,
                                                      unsigned long long* __restrict__ seg) {
  const int r = blockIdx.x * blockDim.x + threadIdx.x;
  if (r >= n_rec || count[r] == 0 || hdr->n_keys == 0ull) return;
  const uint2 rc = rect[r];
  const int tx0 = rc.x & 0xFFFF, ty0 = rc.x >> 16, tx1 = rc.y & 0xFFFF, ty1 = rc.y >> 16;
  const unsigned long long key = ((unsigned long long)depth_bits[r] << 32) | (uint32_t)r;
  for (int ty = ty0; ty < ty1; ++ty)
    for (int tx = tx0; tx < tx1; ++tx) seg[atomicAdd(tile_cursor + ty * TX + tx, 1u)] = key;
}

// ------------------------------------------------------------------------------------------------
// K3: one CTA per tile sorts the tile's segment by (depth bits, record id) — keys are unique, so any correct sort
// gives the one canonical order.  In shared memory when the segment fits (kSortSmemKeys), otherwise in place in
// global memory (a tile with more than 4096 records: rare, and only slower; global writes of a step are visible to
// the CTA's other threads after the barrier).  Writes the canonical arrays of the frame.
constexpr int kSortThreads = 512;
constexpr int kSortSmemKeys = 4096;

// Bitonic sorting network in its all-ascending form (the first step of every merge compares mirrored partners,
// the remaining steps are half-cleaners), over np2 = the next power of two >= n virtual elements of which those at
// index >= n are +infinity.  Every compare-exchange puts the smaller key at the lower index, so a pair whose upper
// index is >= n is a no-op and is skipped: the n real keys are sorted in place for any n.
__device__ __forceinline__ void bitonic_sort(unsigned long long* a, uint32_t n, uint32_t np2) {
  for (uint32_t size = 2; size <= np2; size <<= 1) {
    for (uint32_t stride = size >> 1; stride > 0; stride >>= 1) {
      const bool mirror = stride == (size >> 1);
      for (uint32_t t = threadIdx.x; t < (np2 >> 1); t += kSortThreads) {
        uint32_t lo, hi;
        if (mirror) {
          const uint32_t blk = t / stride, j = t - blk * stride;
          lo = blk * size + j;
          hi = blk * size + size - 1u - j;
        } else {
          lo = 2u * t - (t & (stride - 1u));
          hi = lo + stride;
        }
        if (hi < n) {
          const unsigned long long ka = a[lo], kb = a[hi];
          if (ka > kb) { a[lo] = kb; a[hi] = ka; }
        }
      }
      __syncthreads();
    }
  }
}

// ------------------------------------------------------------------------------------------------
// Render list: the tile's sorted superset list without the records whose conservative q <= tau box touches
// no pixel of the tile — they contribute to no pixel in any state, and every one of the
// ~B/S CTAs that composite the tile would otherwise fetch and drop them again.  Order is kept (ballot
// compaction); the canonical key lists (vals[0], tile_range) are untouched.  Run by the CTA that has just sorted the tile (k_tile_sort).
// The same pass writes the four per-QUADRANT lists the quadrant compositor walks (k_composite_q.cu): quadrant
// (qx, qy) of the tile = the 8x4 blocks qx + 4 qy and qx + 4 qy + 2; its list holds, in depth order, {record id,
// meta} of the records whose block mask has one of the two bits.  The lists of tile t start at 4 * (start of
// t's canonical list) — a tile with n entries owns 4 n slots, n per quadrant — so no allocation pass is needed.
template <int THREADS>
__device__ __forceinline__ void tile_render_lists(int tile, uint2 rg, const unsigned long long* sorted,
                                                  const float4* __restrict__ r0, const float4* __restrict__ r1,
                                                  const float4* __restrict__ rc0, const float4* __restrict__ rc1,
                                                  int TX, uint32_t* __restrict__ rvals,
                                                  uint2* __restrict__ render_range, uint2* __restrict__ qlist,
                                                  uint2* __restrict__ qrange) {
  __shared__ uint32_t s_cnt[THREADS / 32];
  __shared__ uint32_t s_run;
  __shared__ uint32_t s_qcnt[4][THREADS / 32];
  __shared__ uint32_t s_qrun[4];
  const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
  if (tid == 0) s_run = 0;
  if (tid < 4) s_qrun[tid] = 0;
  const uint32_t n_tile = rg.y - rg.x;
  const size_t qbase = 4 * (size_t)rg.x;
  __syncthreads();
  for (uint32_t base = rg.x; base < rg.y; base += THREADS) {
    const uint32_t i = base + tid;
    uint32_t rid = 0, meta = 0;
    uint32_t bm = 0;
    if (i < rg.y) {
      rid = (uint32_t)sorted[i - rg.x];  // low word of (depth bits << 32 | record id)
      const float4 g0 = r0[rid], g1 = r1[rid];
      meta = __float_as_uint(g1.w);
      bm = record_block_mask_tight(g0.x, g0.y, g0.z, g0.w, g1.x, g1.z, rc0[rid].w, rc1[rid].w, tile % TX, tile / TX);
    }
    const bool keep = bm != 0u;
    const uint32_t bal = __ballot_sync(0xffffffffu, keep);
    if (lane == 0) s_cnt[w] = __popc(bal);
    // quadrant q = (q & 1, q >> 1): blocks (q & 1) + 4 (q >> 1) and that + 2
    const uint32_t qm = (bm | (bm >> 2)) & 0x33u;  // bits 0, 1, 4, 5 = quadrants 0, 1, 2, 3
    uint32_t qbal[4];
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      qbal[q] = __ballot_sync(0xffffffffu, (qm >> ((q & 1) + 4 * (q >> 1))) & 1u);
      if (lane == 0) s_qcnt[q][w] = __popc(qbal[q]);
    }
    __syncthreads();
    uint32_t woff = 0, tot = 0;
    for (int q = 0; q < THREADS / 32; ++q) {
      if (q < w) woff += s_cnt[q];
      tot += s_cnt[q];
    }
    if (keep) {
      const uint32_t pos = rg.x + s_run + woff + __popc(bal & ((1u << lane) - 1u));
      rvals[pos] = rid;
    }
    uint32_t qtot[4];
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      uint32_t qoff = 0;
      qtot[q] = 0;
      for (int k = 0; k < THREADS / 32; ++k) {
        if (k < w) qoff += s_qcnt[q][k];
        qtot[q] += s_qcnt[q][k];
      }
      if ((qm >> ((q & 1) + 4 * (q >> 1))) & 1u)
        qlist[qbase + (size_t)q * n_tile + s_qrun[q] + qoff + __popc(qbal[q] & ((1u << lane) - 1u))] = make_uint2(rid, meta);
    }
    __syncthreads();
    if (tid == 0) s_run += tot;
    if (tid < 4) s_qrun[tid] += qtot[tid];
    __syncthreads();
  }
  if (tid == 0) render_range[tile] = make_uint2(rg.x, rg.x + s_run);
  if (tid < 4) {
    const uint32_t st = (uint32_t)(qbase + (size_t)tid * n_tile);
    qrange[4 * tile + tid] = make_uint2(st, st + s_qrun[tid]);
  }
}

__global__ void __launch_bounds__(kSortThreads) k_tile_sort(const uint2* __restrict__ tile_range,
                                                           unsigned long long* __restrict__ seg,
                                                           unsigned long long* __restrict__ keys_out,
                                                           uint32_t* __restrict__ vals_out,
                                                           const float4* __restrict__ r0, const float4* __restrict__ r1,
                                                           const float4* __restrict__ rc0, const float4* __restrict__ rc1,
                                                           int TX, uint32_t* __restrict__ rvals,
                                                           uint2* __restrict__ render_range, uint2* __restrict__ qlist,
                                                           uint2* __restrict__ qrange) {
  __shared__ unsigned long long s_key[kSortSmemKeys];
  const uint32_t tile = blockIdx.x;
  const uint2 rg = tile_range[tile];
  const uint32_t n = rg.y - rg.x;
  if (n == 0) {  // an empty tile still has (empty) render lists
    if (threadIdx.x == 0) render_range[tile] = make_uint2(rg.x, rg.x);
    if (threadIdx.x < 4) qrange[4 * tile + threadIdx.x] = make_uint2(4u * rg.x, 4u * rg.x);
    return;
  }
  uint32_t np2 = 1;
  while (np2 < n) np2 <<= 1;
  unsigned long long* a = seg + rg.x;
  if (n <= kSortSmemKeys) {
    for (uint32_t i = threadIdx.x; i < n; i += kSortThreads) s_key[i] = a[i];
    a = s_key;
    __syncthreads();
  }
  bitonic_sort(a, n, np2);
  for (uint32_t i = threadIdx.x; i < n; i += kSortThreads) {
    const unsigned long long k = a[i];
    keys_out[rg.x + i] = ((unsigned long long)tile << 32) | (k >> 32);
    vals_out[rg.x + i] = (uint32_t)k;
  }
  // a4 preparation while the sorted segment is at hand: render list and the four quadrant lists of the tile
  tile_render_lists<kSortThreads>((int)tile, rg, a, r0, r1, rc0, rc1, TX, rvals, render_range, qlist, qrange);
}

void launch_bin_and_sort(const DeviceScene& sc, const FrameParams& fp, Workspace& ws, long long cap,
                         cudaStream_t st) {
  (void)cap;
  const int n_rec = sc.V * sc.N;
  const int tiles = fp.TX * fp.TY;
  const int grid = (n_rec + 255) / 256;
  k_tile_offsets<<<1, 256, 0, st>>>(ws.tile_cursor, tiles, ws.tile_range, ws.hdr);
  if (n_rec > 0) {
    k_scatter_keys<<<grid, 256, 0, st>>>(n_rec, ws.count, ws.rect, ws.depth_bits, fp.TX, ws.hdr, ws.tile_cursor,
                                         ws.keys[1]);
    k_tile_sort<<<tiles, kSortThreads, 0, st>>>(ws.tile_range, ws.keys[1], ws.keys[0], ws.vals[0], ws.r0, ws.r1, ws.rc0,
                                                ws.rc1, fp.TX, ws.vals[1], ws.render_range, ws.qlist, ws.qrange);
  } else {
    cudaMemsetAsync(ws.render_range, 0, sizeof(uint2) * (size_t)tiles, st);
    cudaMemsetAsync(ws.qrange, 0, sizeof(uint2) * 4 * (size_t)tiles, st);
  }
  count_launches(n_rec > 0 ? 3 : 1);
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
