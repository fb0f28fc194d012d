// k_composite.cu — stage a4 (+ fused a5) of the hot path:
// per-tile front-to-back alpha compositing with early termination, state-blocked.
//
// One CTA = one 16x16 tile x S states of the batch; thread = pixel; each thread keeps (T, r, g, b)
// of its pixel for the S states in registers.  For a record of the tile's depth-sorted superset
// list, alpha of a (pixel, record) pair does NOT depend on the state — only whether the record is
// present does, and that is uniform over the CTA (it depends on the cluster's delivered depth in
// that state).  So alpha is evaluated once and applied to the states in which the record is present:
//     shared by S states : dx, dy, q (spec-exact fp32), the cut q > tau, exp, alpha, 1-alpha
//     per present state  : T' = T(1-alpha); stop if T' < 1e-4; C += alpha T c; T = T'
//
// With tile-level dedup (k_dedup.cu) the S "states" of a CTA are S distinct signature classes of the
// tile; the result is written to every member state of each class.
//
// Staging: the tile's render list (k_tile_render_list: the sorted superset list minus the records that can
// reach no pixel of the tile, with an 8-bit mask of the 8x4 pixel blocks each record can contribute to) is
// gathered 256 entries at a time into shared memory (64 B per record).  A warp owns an 8x4 pixel block; per
// block an ordered list of the staged records whose mask has the block's bit and that are present in at
// least one of the S states is built with warp ballots, so the hot loop only visits records that can matter
// to the warp.  (warp, state) pairs whose 32 pixels have all terminated are retired every 32 records (one
// warp reduction of per-lane liveness masks); the CTA leaves the list when every (pixel, state) is done.
// The per-record tag (which slots contain the record, which take the residual colour) is warp-uniform and
// ptxas knows it (uniform shared addresses), so the slot tests are uniform-datapath skips (ULOP3 + BRA.U).
//
// Determinism: the arithmetic applied to one (pixel, state) is a fixed sequence of explicitly
// rounded fp32 operations that depends only on that state's row of `levels`; skipped work is
// exactly the work that would have been a no-op.  Hence batched == serial bitwise (tests).
#include <atomic>

#include "gsr_internal.h"
#include "reduce.cuh"

namespace gsr {

struct CompositeArgs {
  const uint2* tile_range;
  const uint32_t* vals;
  const uint8_t* vmask;  // per render-list entry: the 8x4 blocks of the tile the record can contribute to
  const float4 *r0, *r1, *rc0, *rc1;
  const int8_t* depth;
  int32_t B, C, nsb;
  int32_t W, H, TX, tiles;
  float bg[3];
  float* out;          // [B,H,W,3] or nullptr
  const float* ref;    // [H,W,3] or nullptr
  double* sse_part;    // [B, tiles]
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

// One (pixel, state) step of DESIGN.md §3.5:  w = alpha T;  T' = T - w  (= T (1 - alpha));  if T' >= 1e-4
// { C += w c; T = T' } else { T = -|T| }.  T < 0 marks a finished pixel (-(frozen transmittance)): then T' <= 0
// and it stays finished.  A lane that failed the cut has alpha = 0, for which the step is exactly a no-op.
// Explicitly rounded (mul.rn / sub.rn / fma.rn, never contracted) and predicated, so that every instantiation
// of the kernel applies bit-identical arithmetic to a state: batched == serial.
// Pipe balance (profiles/r1b): the half-rate ALU pipe (FSETP/FSEL/LOP3) was the binding unit, so the step
// keeps ONE compare and ONE select (with the -|T| folded into its operand) there; the rest is FMA-pipe work.
// T' is formed from the w the colour needs anyway: 7 instructions per state and no 1 - alpha register.
__device__ __forceinline__ void state_update(float& T, float& Cr, float& Cg, float& Cb, float alpha, float cr,
                                             float cg, float cb) {
  asm("{\n\t"
      ".reg .pred p;\n\t"
      ".reg .f32 tn, wg, tm;\n\t"
      "mul.rn.f32 wg, %4, %0;\n\t"
      "sub.rn.f32 tn, %0, wg;\n\t"
      "setp.geu.f32 p, tn, 0f38D1B717;\n\t"  // 1e-4f
      "@p fma.rn.f32 %1, wg, %5, %1;\n\t"
      "@p fma.rn.f32 %2, wg, %6, %2;\n\t"
      "@p fma.rn.f32 %3, wg, %7, %3;\n\t"
      "abs.f32 tm, %0;\n\t"
      "neg.f32 tm, tm;\n\t"
      "selp.f32 %0, tn, tm, p;\n\t"
      "}"
      : "+f"(T), "+f"(Cr), "+f"(Cg), "+f"(Cb)
      : "f"(alpha), "f"(cr), "f"(cg), "f"(cb));
}

__device__ __forceinline__ float ex2_approx_ftz(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}

constexpr float kTStop = 1e-4f;     // reading A11
constexpr float kAlphaCap = 0.99f;  // reading A11

template <int S, bool COUNT>
__global__ void __launch_bounds__(kTilePix, (S <= 8 ? 5 : 2)) k_composite(const CompositeArgs a) {
  extern __shared__ uint16_t s_tab[];  // [C][4]: states (bit s) with depth ==0, >=1, >=2, >=3
  // staged records, 64 B each: {m_x, m_y, A, B} {Cq, tau, -, act | res << 16} {rgb, o} {rgb + SH residual, -}
  __shared__ __align__(16) float4 s_rec[kTilePix * 4];
  __shared__ uint32_t s_lcnt[8][8];            // [list k][source warp]
  __shared__ __align__(16) uint16_t s_list[8][kTilePix];  // per 8x4 block: ordered shared-window addresses of the staged records that touch it
  __shared__ double s_red[8][S];

  const int tid = threadIdx.x, lane = tid & 31;
  const int w = __shfl_sync(0xffffffffu, tid >> 5, 0);  // broadcast: lets the compiler treat the warp index as warp-uniform
  const int tile = blockIdx.x / a.nsb, sb = blockIdx.x - tile * a.nsb;
  const int b0 = sb * S;  // first slot of this block: a state index, or a class index when dedup is on

  // ---- which states this CTA composites.  With tile-level dedup (k_tile_dedup) slot s is the s-th
  //      distinct signature class of this tile from b0 on; its first member stands for the class.
  __shared__ int s_rep[S];        // representative state of slot s, -1 = empty slot
  __shared__ uint32_t s_mlo[S], s_mhi[S];  // members of the class: uorder[tile*B + [mlo, mhi))
  const int n_slots = a.n_unique ? (int)a.n_unique[tile] : a.B;
  if (b0 >= n_slots) return;
  if (tid < S) {
    const int u = b0 + tid;
    int rep = -1;
    uint32_t lo = 0, hi = 0;
    if (u < n_slots) {
      if (a.n_unique) {
        lo = a.upos[(size_t)tile * a.B + u];
        hi = u + 1 < n_slots ? a.upos[(size_t)tile * a.B + u + 1] : (uint32_t)a.B;
        rep = (int)a.uorder[(size_t)tile * a.B + lo];
      } else {
        rep = u;
      }
    }
    s_rep[tid] = rep; s_mlo[tid] = lo; s_mhi[tid] = hi;
  }
  __syncthreads();

  // ---- presence masks of this state block (a0: closure predicates)
  for (int c = tid; c < a.C; c += kTilePix) {
    uint32_t eq0 = 0, ge1 = 0, ge2 = 0, ge3 = 0;
#pragma unroll
    for (int s = 0; s < S; ++s) {
      if (s_rep[s] >= 0) {
        const int d = a.depth[(size_t)s_rep[s] * a.C + c];
        eq0 |= (uint32_t)(d == 0) << s;
        ge1 |= (uint32_t)(d >= 1) << s;
        ge2 |= (uint32_t)(d >= 2) << s;
        ge3 |= (uint32_t)(d >= 3) << s;
      }
    }
    s_tab[4 * c + 0] = (uint16_t)eq0;
    s_tab[4 * c + 1] = (uint16_t)ge1;
    s_tab[4 * c + 2] = (uint16_t)ge2;
    s_tab[4 * c + 3] = (uint16_t)ge3;
  }

  const int tx = tile % a.TX, ty = tile / a.TX;
  // warp w owns the 8x4 pixel block (w & 1, w >> 1) of the tile: compact footprints make the warp-level
  // culls below sharper than 16x2 strips
  const int x = tx * kTile + 8 * (w & 1) + (lane & 7), y = ty * kTile + 4 * (w >> 1) + (lane >> 3);
  const bool inside = x < a.W && y < a.H;
  float px = (float)x + 0.5f, py = (float)y + 0.5f;
  asm volatile("" : "+f"(px), "+f"(py));  // keep them in registers (the compiler would rebuild them per record)
  uint32_t rec_base = (uint32_t)__cvta_generic_to_shared(s_rec);
  uint32_t lbase = (uint32_t)__cvta_generic_to_shared(&s_list[w][0]);
  asm volatile("" : "+r"(rec_base), "+r"(lbase));  // loop-invariant: keep them in registers
  const uint32_t lcnt_base = (uint32_t)__cvta_generic_to_shared(s_lcnt);
  const float bg0 = a.bg[0], bg1 = a.bg[1], bg2 = a.bg[2];

  float T[S], Cr[S], Cg[S], Cb[S];
#pragma unroll
  for (int s = 0; s < S; ++s) {
    T[s] = (inside && s_rep[s] >= 0) ? 1.0f : -1.0f;  // T < 0 marks a finished (pixel, state): -(frozen T)
    Cr[s] = Cg[s] = Cb[s] = 0.0f;
  }

  const uint2 rg = a.tile_range[tile];
  unsigned long long n_shared = 0, n_state = 0, n_logical = 0;  // COUNT only
  __syncthreads();

  for (uint32_t base = rg.x; base < rg.y; base += kTilePix) {
    // ---- stage up to 256 records; drop those present in no state of the block and those whose
    //      q <= tau region (conservative box from k_project) misses the tile
    const uint32_t idx = base + tid;
    const bool have = idx < rg.y;
    // The record keeps slot `tid` of the staging buffer and is written there at once, so that only its block
    // mask stays live across the ballots (the 32 state registers leave little room: profiles/r1j showed the
    // staging spilling to local memory when the four float4 were carried through the compaction).
    uint32_t wmask = 0;
    if (have) {
      const uint32_t rid = __ldg(a.vals + idx);
      const float4 g1 = __ldg(a.r1 + rid);
      const uint32_t meta = __float_as_uint(g1.w);
      const uint32_t cls = meta >> 16;
      const uint16_t* t = s_tab + 4 * (meta & 0xFFFFu);
      uint32_t act, res;
      if (cls >= 16) {
        // 4-variant scene (reading I1): variant v = cls - 16 is present exactly at depth v; only v = 3 has the
        // SH residual colour (stored in both colour slots, so `res` is irrelevant: keep it 0)
        const uint32_t v = cls - 16;
        act = v == 0 ? t[0] : (v == 1 ? (t[1] & ~t[2]) : (v == 2 ? (t[2] & ~t[3]) : t[3]));
        res = 0u;
      } else {
        act = cls == 0 ? t[0] : (cls <= 2 ? t[1] : (cls == 3 ? t[2] : t[3]));
        res = cls == 0 ? 0u : t[3];
      }
      // which 8x4 blocks the record can contribute to was decided once per frame (k_tile_render_list: box, then
      // the minimum of q over the block); records present in no slot of this CTA are not fetched any further
      if (act != 0) wmask = __ldg(a.vmask + idx);
      if (wmask != 0) {
        s_rec[4 * tid + 0] = __ldg(a.r0 + rid);
        s_rec[4 * tid + 1] = make_float4(g1.x, g1.z, 0.0f, __uint_as_float(act | (res << 16)));
        const float4 c0 = __ldg(a.rc0 + rid);
        s_rec[4 * tid + 2] = make_float4(c0.x, c0.y, c0.z, g1.y);
        s_rec[4 * tid + 3] = __ldg(a.rc1 + rid);
      }
    }
    // ordered compaction: each 8x4 pixel block k gets the ordered list s_list[k] of the slots whose region
    // touches it (warp ballots + an 8x8 count table); the ballots are re-taken after the barrier rather than
    // kept in eight registers
    {
      uint32_t cnt = 0;
#pragma unroll
      for (int k = 0; k < 8; ++k) {
        const uint32_t bal = __ballot_sync(0xffffffffu, (wmask >> k) & 1u);
        cnt = lane == k ? __popc(bal) : cnt;
      }
      if (lane < 8) sts32(lcnt_base + 4u * (8u * lane + w), cnt);  // lane k publishes the count of list k
    }
    __syncthreads();
    // exclusive offsets of the 8 source warps inside each of the 8 lists: lane l scans list k = l >> 2, source
    // warps 2 (l & 3) and 2 (l & 3) + 1 (a 4-lane segmented scan), then every lane fetches the offset of ITS
    // warp in list k from lane 4 k + (w >> 1) — 2 shared loads and 10 shuffles instead of an 8 x 8 table walk
    uint32_t nb;  // length of this warp's list
    {
      const uint32_t lk = (uint32_t)lane >> 2, lq = 2u * ((uint32_t)lane & 3u);
      const uint32_t v0 = s_lcnt[lk][lq], v1 = s_lcnt[lk][lq + 1];
      uint32_t incl = v0 + v1;
#pragma unroll
      for (int o = 1; o < 4; o <<= 1) {
        const uint32_t up = __shfl_up_sync(0xffffffffu, incl, o, 4);
        if ((lane & 3) >= o) incl += up;
      }
      const uint32_t off0 = incl - (v0 + v1), off1 = off0 + v0;
      const uint32_t mine = (w & 1) ? off1 : off0;
      nb = __shfl_sync(0xffffffffu, incl, 4 * w + 3);
      const uint32_t lt = (1u << lane) - 1u, mine_addr = rec_base + 64u * tid;
      const uint32_t list0 = lbase - 2u * kTilePix * w;  // shared address of s_list[0][0]
#pragma unroll
      for (int k = 0; k < 8; ++k) {
        const uint32_t off = __shfl_sync(0xffffffffu, mine, 4 * k + (w >> 1));
        const uint32_t bal = __ballot_sync(0xffffffffu, (wmask >> k) & 1u);
        if ((wmask >> k) & 1u) sts16(list0 + 2u * (kTilePix * k + off + __popc(bal & lt)), mine_addr);
      }
    }
    __syncthreads();

    // ---- composite this warp's records in order
    for (uint32_t j0 = 0; j0 < nb; j0 += 32u) {
      // refresh the (warp, slot) liveness mask every 32 records
      uint32_t walive = 0;
#pragma unroll
      for (int s = 0; s < S; ++s) walive |= (T[s] > 0.0f ? 1u : 0u) << s;
      walive = __reduce_or_sync(0xffffffffu, walive);  // one warp reduction of the per-lane masks instead of S votes
      if (walive == 0) break;
      const uint32_t j1 = min(nb, j0 + 32u);
#pragma unroll 2
      for (uint32_t j = j0; j < j1; ++j) {
        const uint32_t addr = lds16(lbase + 2u * j);
        const float4 hq = lds128(addr + 16u);  // {Cq, tau, -, act | res << 16}
        const uint32_t tag = __float_as_uint(hq.w);
        const uint32_t actl = tag & walive;  // slots that contain the record and are still alive
        // (a record left with no live slot, 2 % of the iterations on cfg1, is not skipped: the test costs more
        //  than the no-op iterations it saves — measured on cfg1, cfg2 and cfg4)
        const float4 h0 = lds128(addr);
        const float2 h1 = make_float2(hq.x, hq.y);  // {Cq, tau}
        // spec-exact quadratic form: u = A dx; s = fma(B,dy,u); q = s dx; v = Cq dy; q = fma(v,dy,q)
        const float dx = __fsub_rn(h0.x, px);
        const float dy = __fsub_rn(h0.y, py);
        const float u = __fmul_rn(h0.z, dx);
        const float sacc = __fmaf_rn(h0.w, dy, u);
        float q = __fmul_rn(sacc, dx);
        const float v = __fmul_rn(h1.x, dy);
        q = __fmaf_rn(v, dy, q);
        const bool pass = !(q > h1.y);  // skip iff q > tau  (alpha < 1/255)
        if (COUNT) {
          int live = 0, logical = 0;
#pragma unroll
          for (int s = 0; s < S; ++s) {
            const bool l = ((actl >> s) & 1u) && T[s] > 0.0f;
            live += l;
            logical += l ? (a.n_unique ? (int)(s_mhi[s] - s_mlo[s]) : 1) : 0;  // every member of the class
          }
          n_shared += live > 0;
          n_logical += logical;
          n_state += pass ? live : 0;
        }
        // (no warp vote here: after the per-block q_min culling of k_tile_render_list a record whose cut fails on
        //  all 32 pixels reaches this point in 0.3 % of the iterations; alpha = 0 makes the updates no-ops)
        const float4 k0 = lds128(addr + 32u);
        // q <= tau <= ln 255 on every lane that passes: no denormal range to guard, ex2.approx.ftz is enough
        float alpha = fminf(kAlphaCap, __fmul_rn(k0.w, ex2_approx_ftz(__fmul_rn(q, -1.4426950408889634f))));
        alpha = pass ? alpha : 0.0f;
        // The tag is the same on every lane, and ptxas knows it: the list entry and the record are loaded from
        // warp-uniform shared addresses, so the tag lands in a uniform register (R2UR) and every slot test below
        // is a plain uniform skip (BRA.U) without reconvergence barriers — no warp reduction needed to say so.
        // Slots taking the plain colour first, then those taking the colour with the SH residual.
        const uint32_t act1 = actl & (tag >> 16), act0 = actl ^ act1;
#pragma unroll
        for (int s = 0; s < S; ++s)
          if ((act0 >> s) & 1u) state_update(T[s], Cr[s], Cg[s], Cb[s], alpha, k0.x, k0.y, k0.z);
        if (act1 != 0) {
          const float4 k1 = lds128(addr + 48u);
#pragma unroll
          for (int s = 0; s < S; ++s)
            if ((act1 >> s) & 1u) state_update(T[s], Cr[s], Cg[s], Cb[s], alpha, k1.x, k1.y, k1.z);
        }
      }
    }
    bool any_alive = false;
#pragma unroll
    for (int s = 0; s < S; ++s) any_alive |= T[s] > 0.0f;
    if (base + kTilePix >= rg.y) break;  // last chunk: nothing left to stage, no need to meet the other warps
    if (!__syncthreads_or(any_alive)) break;
  }

  if (COUNT) {
    n_shared = (unsigned long long)warp_sum_butterfly((double)n_shared);
    n_state = (unsigned long long)warp_sum_butterfly((double)n_state);
    n_logical = (unsigned long long)warp_sum_butterfly((double)n_logical);
    if (lane == 0) {
      atomicAdd(a.counts + 0, n_shared);
      atomicAdd(a.counts + 1, n_state);
      atomicAdd(a.counts + 2, n_logical);
    }
    return;
  }
  // ---- pixel = C + T * background; optional fused squared error against the reference
  float rr0 = 0.f, rr1 = 0.f, rr2 = 0.f;
  if (a.ref && inside) {
    const float* rp = a.ref + ((size_t)y * a.W + x) * 3;
    rr0 = __ldg(rp); rr1 = __ldg(rp + 1); rr2 = __ldg(rp + 2);
  }
  // the squared errors stay in fp32 registers until the reduction (the widening is exact); the image pointer of
  // a member state is one 32 x 32 -> 64-bit multiply-add from the pixel's pointer in image 0
  float errf[S];
  float* const pixp = a.out ? a.out + ((size_t)y * a.W + x) * 3 : nullptr;
  const uint32_t img = (uint32_t)a.H * (uint32_t)a.W * 3u;  // floats per image (< 2^32: checked by camera_ok at the API)
  const uint32_t* const mem = a.n_unique ? a.uorder + (size_t)tile * a.B : nullptr;
#pragma unroll
  for (int s = 0; s < S; ++s) {
    const float Tf = fabsf(T[s]);  // the transmittance the pixel ended with (frozen at termination)
    const float o0 = __fmaf_rn(Tf, bg0, Cr[s]);
    const float o1 = __fmaf_rn(Tf, bg1, Cg[s]);
    const float o2 = __fmaf_rn(Tf, bg2, Cb[s]);
    if (a.out && inside && s_rep[s] >= 0) {
      // every state of the class receives the (identical) tile; without dedup the "class" is the state itself.
      // One loop for both and not unrolled: the epilogue is instantiated per slot and its code size costs
      // instruction-cache hits of the record loop (measured: -1.2 % kernel time for the rolled loop)
      const uint32_t lo = mem ? s_mlo[s] : (uint32_t)s_rep[s], hi = mem ? s_mhi[s] : lo + 1u;
#pragma unroll 1
      for (uint32_t i = lo; i < hi; ++i) {
        float* op = pixp + (size_t)(mem ? __ldg(mem + i) : i) * img;
        __stcs(op, o0); __stcs(op + 1, o1); __stcs(op + 2, o2);  // write-once stream: evict first
      }
    }
    errf[s] = (a.ref && inside) ? pixel_sq_err(o0, o1, o2, rr0, rr1, rr2) : 0.0f;
  }
  if (a.ref) {
    int slot;
    double err[S];
#pragma unroll
    for (int s = 0; s < S; ++s) err[s] = (double)errf[s];
    const double tot = warp_sum_slots<S>(err, lane, slot);  // same bits as S plain butterflies (reduce.cuh)
    if ((lane & (32 / S - 1)) == 0) s_red[w][slot] = tot;
    __syncthreads();
    if (tid < S && s_rep[tid] >= 0) {
      double acc = s_red[0][tid];
#pragma unroll
      for (int k = 1; k < 8; ++k) acc += s_red[k][tid];
      if (a.n_unique) {
        const uint32_t* mem = a.uorder + (size_t)tile * a.B;
        for (uint32_t i = s_mlo[tid]; i < s_mhi[tid]; ++i) a.sse_part[(size_t)mem[i] * a.tiles + tile] = acc;
      } else {
        a.sse_part[(size_t)s_rep[tid] * a.tiles + tile] = acc;
      }
    }
  }
}

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

int g_state_block = 8;  // S; set through gsr_set_option for experiments (1, 4, 8, 16)
int g_dedup = 1;        // gsr_set_option("dedup", 0/1): tile-level state dedup
int g_profile = 0;      // gsr_set_option("profile", 1): record events around every k_composite launch
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

template <int S, bool COUNT>
static void launch_composite_S(const CompositeArgs& a, cudaStream_t st) {
  const size_t smem = sizeof(uint16_t) * 4 * (size_t)a.C;
  const long long grid = (long long)a.tiles * a.nsb;
  static bool attr_set = false;  // per instantiation: static + dynamic shared memory passes 48 KB from C ~ 3300 on
  if (!attr_set) {
    cudaFuncSetAttribute(k_composite<S, COUNT>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                         (int)(sizeof(uint16_t) * 4 * kMaxC));
    attr_set = true;
  }
  int slot = -1;
  if (!COUNT && g_profile && g_ev_used < kMaxProfEvents) {
    slot = g_ev_used++;
    while (g_ev_created <= slot) {
      cudaEventCreate(&g_ev[g_ev_created][0]);
      cudaEventCreate(&g_ev[g_ev_created][1]);
      ++g_ev_created;
    }
    cudaEventRecord(g_ev[slot][0], st);
  }
  k_composite<S, COUNT><<<(unsigned)grid, kTilePix, smem, st>>>(a);
  if (slot >= 0) cudaEventRecord(g_ev[slot][1], st);
  count_launches(1);
}

static CompositeArgs make_args(const DeviceScene& sc, const FrameParams& fp, Workspace& ws, const int8_t* depth_rows,
                               int32_t B) {
  CompositeArgs a;
  a.tile_range = ws.render_range;  // the render list: sorted superset list minus the sub-tile-culled records
  a.vals = ws.vals[1];
  a.vmask = (const uint8_t*)ws.keys[1];
  a.r0 = ws.r0; a.r1 = ws.r1; a.rc0 = ws.rc0; a.rc1 = ws.rc1;
  a.depth = depth_rows;
  a.B = B; a.C = sc.C;
  a.W = fp.W; a.H = fp.H; a.TX = fp.TX; a.tiles = fp.TX * fp.TY;
  a.bg[0] = fp.bg[0]; a.bg[1] = fp.bg[1]; a.bg[2] = fp.bg[2];
  a.out = nullptr; a.ref = nullptr; a.sse_part = ws.sse_part; a.counts = nullptr;
  a.uorder = nullptr; a.upos = nullptr; a.n_unique = nullptr;
  return a;
}

template <bool COUNT>
static void dispatch_composite(CompositeArgs& a, cudaStream_t st) {
  int S = g_state_block;
  if (a.B == 1) S = 1;
  a.nsb = (a.B + S - 1) / S;
  switch (S) {
    case 1: launch_composite_S<1, COUNT>(a, st); break;
    case 4: launch_composite_S<4, COUNT>(a, st); break;
    case 16: launch_composite_S<16, COUNT>(a, st); break;
    default: launch_composite_S<8, COUNT>(a, st); break;
  }
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
    a.sse_part = ws.sse_part + (size_t)b0 * tiles;
    if (g_dedup && launch_tile_dedup(sc, fp, ws, rows, nb, st)) {
      a.uorder = ws.uorder; a.upos = ws.upos; a.n_unique = ws.n_unique;
    }
    dispatch_composite<false>(a, st);
  }
  if (ref) launch_distortion_finalize(ws.sse_part, B, tiles, (int64_t)3 * fp.W * fp.H, mse, psnr, st);
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

}  // namespace gsr
