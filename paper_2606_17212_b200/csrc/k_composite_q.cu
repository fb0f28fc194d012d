// k_composite_q.cu — stage a4 (+ fused a5), quadrant compositor.
//
// One CTA = ONE WARP = one 8x8 pixel quadrant of a tile x S state slots.  A lane owns TWO pixels — (x, y) in the
// upper 8x4 block of the quadrant and (x, y + 4) in the lower one — and keeps (T, r, g, b) of both for the S
// slots in 64-bit register pairs, so that every floating-point step of the hot loop is ONE packed instruction
// for the two pixels (Blackwell fma/mul/add.rn.f32x2: SASS FFMA2 / FMUL2 / FADD2; each half is an independent
// IEEE round-to-nearest operation).  Whether a slot contains a record is a property of the slot, i.e. the same
// for both halves of the pair: the packed lanes are dense (pairing two SLOTS instead was measured: 1.4 of the 2
// halves useful, no gain — DESIGN.md §15).
//
//     shared by the S slots : dx, dy, q (spec-exact fp32), the cut q > tau, exp, alpha     (packed: 2 pixels)
//     per present slot      : w = alpha T; T = T - w; s = [T >= 1e-4]; C += (s w)(c - bg)   (packed: 2 pixels)
//
// Stop rule without a select: T keeps decaying after the stop and alpha >= 0 makes it non-increasing, so once
// T < 1e-4 every later s is 0 and nothing is added any more (s is taken from the NEW T: "this Gaussian is not
// added").  The frozen transmittance is not needed: pixel = C + T_stop bg with T_stop = 1 - sum of the accepted
// w, hence pixel = bg + sum (s w)(c - bg); k_project stores c - bg in the packed records.  T, w and C are carried scaled by 2^40
// (exact), which makes the step ONE saturating add with an immediate: s = sat(2^40 T - 2^40 pred(1e-4)):
// neighbouring floats at 1e-4 are 2^-37 apart, so T >= 1e-4 gives >= 8 -> 1 and T <= pred(1e-4) gives <= 0 -> 0.
//
// No barrier anywhere: the warp walks the quadrant's own render list (k_tile_sort, once per frame: the
// tile's depth-sorted list restricted to the records whose q <= tau region can reach the quadrant), 32 entries
// at a time: each lane takes one entry {record id, meta}, derives from the presence table which of the S slots
// contain the record, and the records present in at least one slot are copied global -> shared with cp.async
// (64 bytes each, compacted in list order by a ballot) into one of two buffers while the previous chunk is being
// composited.  The tag of a staged record (slots that contain it, slots that take the residual colour) is
// warp-uniform and read from a uniform shared address, so the slot tests are uniform-datapath skips.
//
// Determinism: the arithmetic applied to one (pixel, state) is a fixed sequence of explicitly rounded fp32
// operations that depends only on that state's row of `levels`; skipped work is exactly the work that would
// have been a no-op.  Hence batched == serial bitwise (tests).
#include "composite_common.cuh"
#include "gsr_internal.h"
#include "reduce.cuh"

namespace gsr {

// One slot, two pixels: DESIGN.md §3.5 in the scaled form of the header.  8 instructions, all on the FMA pipe.
__device__ __forceinline__ void slot_update(f32x2& T, f32x2& Cr, f32x2& Cg, f32x2& Cb, f32x2 alpha2, float cr,
                                            float cg, float cb) {
  asm("{\n\t"
      ".reg .b64 w, s, c;\n\t"
      ".reg .f32 tl, th;\n\t"
      "mul.rn.f32x2 w, %4, %0;\n\t"
      "sub.rn.f32x2 %0, %0, w;\n\t"
      "mov.b64 {tl, th}, %0;\n\t"
      "add.rn.sat.f32 tl, tl, 0fCCD1B716;\n\t"  // -pred(1e-4f) 2^40
      "add.rn.sat.f32 th, th, 0fCCD1B716;\n\t"
      "mov.b64 s, {tl, th};\n\t"
      "mul.rn.f32x2 w, w, s;\n\t"
      "mov.b64 c, {%5, %5};\n\t"
      "fma.rn.f32x2 %1, w, c, %1;\n\t"
      "mov.b64 c, {%6, %6};\n\t"
      "fma.rn.f32x2 %2, w, c, %2;\n\t"
      "mov.b64 c, {%7, %7};\n\t"
      "fma.rn.f32x2 %3, w, c, %3;\n\t"
      "}"
      : "+l"(T), "+l"(Cr), "+l"(Cg), "+l"(Cb)
      : "l"(alpha2), "f"(cr), "f"(cg), "f"(cb));
}

constexpr int kRecordUnroll = 2;

template <int S, bool COUNT>
__global__ void __launch_bounds__(32, (S <= 5 ? 32 : (S <= 6 ? 28 : (S <= 8 ? 24 : 5)))) k_composite_q(const CompositeArgs a) {
  extern __shared__ uint16_t s_tab[];  // [C][4]: slots (bit s) whose state has depth == 0, >= 1, >= 2, >= 3
  __shared__ __align__(16) float4 s_rec[2][kChunk * 4];  // two staging buffers of 32 packed records
  __shared__ uint32_t s_tag[2][kChunk];                  // act | res << 16 of the staged records
  __shared__ int s_rep[S];                 // representative state of slot s, -1 = empty slot
  __shared__ uint32_t s_mlo[S], s_mhi[S];  // members of the class: uorder[tile*B + [mlo, mhi))

  const int lane = threadIdx.x;
  // Persistent warps: the grid is one wave of one-warp CTAs and every warp takes work items — (tile, quadrant,
  // state block) in launch order — from a counter until none is left, so that a register slot is never empty
  // between two CTAs (one-warp CTAs live ~30 us; the launch gap showed as 5.5 of 7 warps resident).
  for (;;) {
  uint32_t item = 0;
  if (lane == 0) item = atomicAdd(a.work_counter, 1u);
  item = __shfl_sync(0xffffffffu, item, 0);
  if (item >= a.n_items) break;
  const uint32_t tq = item / (uint32_t)a.nsb;  // 4 * tile + quadrant
  const int sb = (int)(item - tq * (uint32_t)a.nsb);
  const int tile = (int)(tq >> 2), quad = (int)(tq & 3u);
  const int b0 = sb * S;  // first slot of this block: a state index, or a class index when dedup is on

  // ---- which states this warp composites.  With tile-level dedup (k_tile_dedup) slot s is the s-th distinct
  //      signature class of this tile from b0 on; its first member stands for the class.
  const int n_slots = a.n_unique ? (int)a.n_unique[tile] : a.B;
  if (b0 >= n_slots) continue;
  if (lane < S) {
    const int u = b0 + lane;
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
    s_rep[lane] = rep; s_mlo[lane] = lo; s_mhi[lane] = hi;
  }
  __syncwarp();

  // ---- presence masks of this state block (a0: closure predicates)
  for (int c = lane; c < a.C; c += 32) {
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
  __syncwarp();

  const int tx = tile % a.TX, ty = tile / a.TX;
  const uint32_t rec_base = (uint32_t)__cvta_generic_to_shared(&s_rec[0][0]);
  const uint32_t tag_base = (uint32_t)__cvta_generic_to_shared(&s_tag[0][0]);
  const uint32_t lt = (1u << lane) - 1u;
  unsigned long long n_shared = 0, n_state = 0, n_logical = 0;  // COUNT only
  // quadrant (qx, qy) of tile (tx, ty): the 8x4 blocks k0 = qx + 4 qy (rows 8 qy ..) and k0 + 2 (rows 8 qy + 4 ..)
  const int x = tx * kTile + 8 * (quad & 1) + (lane & 7);
  const int ya = ty * kTile + 8 * (quad >> 1) + (lane >> 3), yb = ya + 4;
  const bool in_a = x < a.W && ya < a.H, in_b = x < a.W && yb < a.H;
  float px = (float)x + 0.5f;
  f32x2 npy2 = pack2(-((float)ya + 0.5f), -((float)yb + 0.5f));  // m_y - p_y == m_y + (-p_y) bit for bit
  asm volatile("" : "+f"(px), "+l"(npy2));  // keep them in registers (the compiler would rebuild them per record)

  // slot s: lo half = the pixel of the upper block, hi half = the pixel of the lower block; an empty slot or a
  // pixel outside the image starts with T = 0, for which every step is a no-op
  f32x2 T2[S], Cr2[S], Cg2[S], Cb2[S];
#pragma unroll
  for (int s = 0; s < S; ++s) {
    const bool on = s_rep[s] >= 0;
    T2[s] = pack2(on && in_a ? kTScale : 0.0f, on && in_b ? kTScale : 0.0f);
    Cr2[s] = Cg2[s] = Cb2[s] = pack2(0.0f, 0.0f);
  }

  const uint2 qr = a.qrange[tq];
  const uint32_t n_ent = qr.y - qr.x;
  const uint2* const list = a.qlist + qr.x;

  // stage one chunk: the lane's entry -> slots that contain the record -> cp.async of the kept records
  auto stage = [&](uint2 e, bool have, int buf) -> uint32_t {
    uint32_t act = 0, res = 0;
    if (have) {
      const uint32_t meta = e.y, cls = meta >> 16;
      const uint16_t* t = s_tab + 4 * (meta & 0xFFFFu);
      if (cls >= 16) {
        // 4-variant scene (reading I1): variant v = cls - 16 is present exactly at depth v; only v = 3 has the
        // SH residual colour (stored in both colour slots, so `res` is irrelevant: keep it 0)
        const uint32_t v = cls - 16;
        act = v == 0 ? t[0] : (v == 1 ? (t[1] & ~t[2]) : (v == 2 ? (t[2] & ~t[3]) : t[3]));
      } else {
        act = cls == 0 ? t[0] : (cls <= 2 ? t[1] : (cls == 3 ? t[2] : t[3]));
        res = cls == 0 ? 0u : t[3];
      }
    }
    const bool keep = act != 0;
    const uint32_t bal = __ballot_sync(0xffffffffu, keep);
    if (keep) {
      const uint32_t pos = __popc(bal & lt);
      const uint32_t dst = rec_base + (uint32_t)buf * (kChunk * 64u) + 64u * pos;
      const float4* src = a.rec + 4 * (size_t)e.x;
      cp_async16(dst, src);
      cp_async16(dst + 16u, src + 1);
      cp_async16(dst + 32u, src + 2);
      cp_async16(dst + 48u, src + 3);
      sts32(tag_base + (uint32_t)buf * (kChunk * 4u) + 4u * pos, act | (res << 16));
    }
    cp_async_commit();
    return (uint32_t)__popc(bal);
  };

  uint32_t n_cur = 0;
  uint2 e_next = make_uint2(0u, 0u);
  if (n_ent > 0) {
    const uint2 e0 = (uint32_t)lane < n_ent ? __ldg(list + lane) : make_uint2(0u, 0u);
    n_cur = stage(e0, (uint32_t)lane < n_ent, 0);
    if (kChunk + (uint32_t)lane < n_ent) e_next = __ldg(list + kChunk + lane);
  }

  for (uint32_t base = 0; base < n_ent; base += kChunk) {
    const int buf = (int)((base / kChunk) & 1u);
    // the next chunk goes to the other buffer while this one is composited (every lane has left that buffer:
    // the warp met at the __syncwarp below one round ago)
    uint32_t n_nxt = 0;
    const bool more = base + kChunk < n_ent;
    if (more) {
      n_nxt = stage(e_next, base + kChunk + (uint32_t)lane < n_ent, buf ^ 1);
      if (base + 2 * kChunk + (uint32_t)lane < n_ent) e_next = __ldg(list + base + 2 * kChunk + lane);
      cp_async_wait<1>();
    } else {
      cp_async_wait<0>();
    }
    __syncwarp();

    // refresh the (warp, slot) liveness mask once per chunk
    uint32_t walive = 0;
#pragma unroll
    for (int s = 0; s < S; ++s) {
      float t0, t1;
      unpack2(T2[s], t0, t1);
      walive |= ((t0 >= kTStopScaled || t1 >= kTStopScaled) ? 1u : 0u) << s;
    }
    walive = __reduce_or_sync(0xffffffffu, walive);
    if (walive == 0) {
      cp_async_wait<0>();
      break;
    }

    const uint32_t rb0 = rec_base + (uint32_t)buf * (kChunk * 64u), tb0 = tag_base + (uint32_t)buf * (kChunk * 4u);
#pragma unroll kRecordUnroll
    for (uint32_t j = 0; j < n_cur; ++j) {
      const uint32_t addr = rb0 + 64u * j;
      const uint32_t tag = lds32(tb0 + 4u * j);
      const uint32_t actl = tag & walive;  // slots that contain the record and are still alive
      const float4 h0 = lds128(addr);        // {m_x, m_y, A, B}
      const float4 hq = lds128(addr + 16u);  // {Cq, tau, o, -}
      // spec-exact quadratic form per pixel: u = A dx; s = fma(B,dy,u); q = s dx; v = Cq dy;
      // q = fma(v,dy,q) — the two pixels share dx
      const float dx = __fsub_rn(h0.x, px);
      const f32x2 dy2 = add2(npy2, pack2(h0.y, h0.y));
      const float u = __fmul_rn(h0.z, dx);
      const f32x2 s2 = fma2(dy2, pack2(h0.w, h0.w), pack2(u, u));
      f32x2 q2 = mul2(s2, pack2(dx, dx));
      const f32x2 v2 = mul2(dy2, pack2(hq.x, hq.x));
      q2 = fma2(v2, dy2, q2);
      float qa, qb;
      unpack2(q2, qa, qb);
      const bool pass_a = !(qa > hq.y), pass_b = !(qb > hq.y);  // skip iff q > tau  (alpha < 1/255)
      if (COUNT) {
        int live_a = 0, live_b = 0, log_a = 0, log_b = 0;
#pragma unroll
        for (int s = 0; s < S; ++s) {
          float t0, t1;
          unpack2(T2[s], t0, t1);
          const int mem = a.n_unique ? (int)(s_mhi[s] - s_mlo[s]) : 1;  // every member of the class
          const bool la = ((actl >> s) & 1u) && t0 >= kTStopScaled, lb = ((actl >> s) & 1u) && t1 >= kTStopScaled;
          live_a += la; live_b += lb;
          log_a += la ? mem : 0; log_b += lb ? mem : 0;
        }
        n_shared += (live_a > 0) + (live_b > 0);
        n_logical += log_a + log_b;
        n_state += (pass_a ? live_a : 0) + (pass_b ? live_b : 0);
      }
      const float4 k0 = lds128(addr + 32u);  // {rgb - bg, -}
      // q <= tau <= ln 255 on every pixel that passes: no denormal range to guard, ex2.approx.ftz is enough
      float al_a = fminf(kAlphaCap, __fmul_rn(hq.z, ex2_approx_ftz(__fmul_rn(qa, -1.4426950408889634f))));
      float al_b = fminf(kAlphaCap, __fmul_rn(hq.z, ex2_approx_ftz(__fmul_rn(qb, -1.4426950408889634f))));
      al_a = pass_a ? al_a : 0.0f;
      al_b = pass_b ? al_b : 0.0f;
      const f32x2 alpha2 = pack2(al_a, al_b);
      // slots taking the plain colour first, then those taking the colour with the SH residual
      const uint32_t act1 = actl & (tag >> 16), act0 = actl ^ act1;
#pragma unroll
      for (int s = 0; s < S; ++s)
        if ((act0 >> s) & 1u) slot_update(T2[s], Cr2[s], Cg2[s], Cb2[s], alpha2, k0.x, k0.y, k0.z);
      if (act1 != 0) {
        const float4 k1 = lds128(addr + 48u);
#pragma unroll
        for (int s = 0; s < S; ++s)
          if ((act1 >> s) & 1u) slot_update(T2[s], Cr2[s], Cg2[s], Cb2[s], alpha2, k1.x, k1.y, k1.z);
      }
    }
    n_cur = n_nxt;
    __syncwarp();  // every lane is done with `buf` before the next round overwrites it
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
    continue;
  }

  // ---- pixel = bg + 2^-40 C (C accumulated relative to the background, scaled); optional fused squared error
  const float bg0 = a.bg[0], bg1 = a.bg[1], bg2 = a.bg[2];
  float ra[3] = {0.f, 0.f, 0.f}, rbv[3] = {0.f, 0.f, 0.f};
  if (a.ref) {
    if (in_a) {
      const float* rp = a.ref + ((size_t)ya * a.W + x) * 3;
      ra[0] = __ldg(rp); ra[1] = __ldg(rp + 1); ra[2] = __ldg(rp + 2);
    }
    if (in_b) {
      const float* rp = a.ref + ((size_t)yb * a.W + x) * 3;
      rbv[0] = __ldg(rp); rbv[1] = __ldg(rp + 1); rbv[2] = __ldg(rp + 2);
    }
  }
  // squared errors: index 2 s + h (h = 0 upper block, 1 lower block); they stay fp32 until the reduction
  float errf[2 * S];
  float* const pix_a = a.out ? a.out + ((size_t)ya * a.W + x) * 3 : nullptr;
  const uint32_t img = (uint32_t)a.H * (uint32_t)a.W * 3u;  // floats per image (< 2^32: checked by camera_ok at the API)
  const uint32_t row4 = 4u * (uint32_t)a.W * 3u;            // the lower pixel sits four rows further down
  const uint32_t* const mem = a.n_unique ? a.uorder + (size_t)tile * a.B : nullptr;
#pragma unroll
  for (int s = 0; s < S; ++s) {
    float cr[2], cg[2], cb[2];
    unpack2(Cr2[s], cr[0], cr[1]);
    unpack2(Cg2[s], cg[0], cg[1]);
    unpack2(Cb2[s], cb[0], cb[1]);
    const float a0 = __fmaf_rn(cr[0], kInvTScale, bg0), a1 = __fmaf_rn(cg[0], kInvTScale, bg1), a2 = __fmaf_rn(cb[0], kInvTScale, bg2);
    const float c0 = __fmaf_rn(cr[1], kInvTScale, bg0), c1 = __fmaf_rn(cg[1], kInvTScale, bg1), c2 = __fmaf_rn(cb[1], kInvTScale, bg2);
    if (a.out && in_a && s_rep[s] >= 0) {
      // every state of the class receives the (identical) pixels; without dedup the "class" is the state itself
      const uint32_t lo = mem ? s_mlo[s] : (uint32_t)s_rep[s], hi = mem ? s_mhi[s] : lo + 1u;
#pragma unroll 1
      for (uint32_t i = lo; i < hi; ++i) {
        float* op = pix_a + (size_t)(mem ? __ldg(mem + i) : i) * img;
        __stcs(op, a0); __stcs(op + 1, a1); __stcs(op + 2, a2);  // write-once stream: evict first
        if (in_b) { __stcs(op + row4, c0); __stcs(op + row4 + 1, c1); __stcs(op + row4 + 2, c2); }
      }
    }
    errf[2 * s] = (a.ref && in_a) ? pixel_sq_err(a0, a1, a2, ra[0], ra[1], ra[2]) : 0.0f;
    errf[2 * s + 1] = (a.ref && in_b) ? pixel_sq_err(c0, c1, c2, rbv[0], rbv[1], rbv[2]) : 0.0f;
  }
  if (a.ref) {
    int slot;
    constexpr int NR = 2 * S <= 2 ? 2 : (2 * S <= 4 ? 4 : (2 * S <= 8 ? 8 : (2 * S <= 16 ? 16 : 32)));  // padded to a power of two
    double err[NR];
#pragma unroll
    for (int k = 0; k < NR; ++k) err[k] = k < 2 * S ? (double)errf[k < 2 * S ? k : 0] : 0.0;
    // per (slot, block) the canonical xor butterfly over the block's 32 pixels (reduce.cuh); the blocks of a tile
    // are added in index order by k_distortion_finalize_blk
    const double tot = warp_sum_slots<NR>(err, lane, slot);
    if ((lane & (32 / NR - 1)) == 0 && slot < 2 * S) {
      const int s = slot >> 1, blk = (quad & 1) + 4 * (quad >> 1) + 2 * (slot & 1);
      if (s_rep[s] >= 0) {
        if (a.n_unique) {
          for (uint32_t i = s_mlo[s]; i < s_mhi[s]; ++i) a.sse_blk[((size_t)mem[i] * a.tiles + tile) * 8 + blk] = tot;
        } else {
          a.sse_blk[((size_t)s_rep[s] * a.tiles + tile) * 8 + blk] = tot;
        }
      }
    }
  }
  __syncwarp();  // the shared tables and buffers are rewritten by the next item
  }
}

// One CTA per state.  The tree is the one of reduce.cuh — per tile the eight block partials in index order, tiles
// lane-strided in index order (lane l adds tiles l, l + 32, ...), then the butterfly — but the per-tile sums are
// formed by all 256 threads first (4096 tiles at a time, in shared memory) and one warp then walks them in that
// order: the same additions in the same order as one warp doing everything, at a fraction of the latency.
constexpr int kFinTiles = 4096;  // a multiple of 32: the lane of a tile does not depend on the chunking
__global__ void __launch_bounds__(256) k_distortion_finalize_blk(const double* __restrict__ blk, int B, int tiles,
                                                                 double inv_n, double* __restrict__ mse,
                                                                 float* __restrict__ psnr) {
  __shared__ double s_tile[kFinTiles];
  const int b = blockIdx.x, lane = threadIdx.x & 31;
  double acc = 0.0;
  for (int base = 0; base < tiles; base += kFinTiles) {
    const int n = min(kFinTiles, tiles - base);
    for (int i = threadIdx.x; i < n; i += 256) {
      const double* p = blk + ((size_t)b * tiles + base + i) * 8;
      double t = p[0];
#pragma unroll
      for (int w = 1; w < 8; ++w) t += p[w];
      s_tile[i] = t;
    }
    __syncthreads();
    if (threadIdx.x < 32)
      for (int k = lane; k < n; k += 32) acc += s_tile[k];
    __syncthreads();
  }
  if (threadIdx.x < 32) {
    acc = warp_sum_butterfly(acc);
    if (lane == 0) {
      const double m = acc * inv_n;
      mse[b] = m;
      if (psnr) psnr[b] = (float)(-10.0 * log10(m > 1e-10 ? m : 1e-10));
    }
  }
}

void launch_distortion_finalize_blk(const double* blk, int32_t B, int32_t tiles, int64_t n_values, double* mse,
                                    float* psnr, cudaStream_t st) {
  if (B == 0) return;
  k_distortion_finalize_blk<<<B, 256, 0, st>>>(blk, B, tiles, 1.0 / (double)n_values, mse, psnr);
  count_launches(1);
}

template <int S, bool COUNT>
static void launch_q_S(const CompositeArgs& a, cudaStream_t st) {
  const size_t smem = sizeof(uint16_t) * 4 * (size_t)a.C;
  const long long items = (long long)a.tiles * 4 * a.nsb;
  if (smem > 40 * 1024)  // static + dynamic shared memory passes 48 KB for very large C
    cudaFuncSetAttribute(k_composite_q<S, COUNT>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                         (int)(sizeof(uint16_t) * 4 * kMaxC));
  // one wave: as many one-warp CTAs as fit the device at this kernel's register and shared-memory use
  int dev = 0, sms = 1, per_sm = 1;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_composite_q<S, COUNT>, 32, smem);
  const long long wave = (long long)sms * (per_sm > 0 ? per_sm : 1);
  CompositeArgs b = a;
  b.n_items = (uint32_t)items;
  cudaMemsetAsync(b.work_counter, 0, sizeof(uint32_t), st);
  const long long grid = items < wave ? items : wave;
  k_composite_q<S, COUNT><<<(unsigned)grid, 32, smem, st>>>(b);
}

// States per warp.  Measured on cfg1 (states/s, 4 frames in flight): S = 4: 78.5 k, 5: 83.7 k, 6: 86.0 k, 7: 78.4 k,
// 8: 84.8 k (80 registers, small spills; 82.5 k at 90 registers).  More slots share one alpha evaluation, fewer
// warps fit: 8 S state registers + ~24 others -> 8 / 7 / 6 / 5 warps per scheduler at S = 5 / 6 / 8 (80) / 8 (90).
constexpr int kDefaultStateBlock = 6;

// S = 0: default
void launch_composite_q(const CompositeArgs& a_in, int S, bool count, cudaStream_t st) {
  CompositeArgs a = a_in;
  if (S == 0) S = kDefaultStateBlock;
  if (a.B == 1) S = 1;
  a.nsb = (a.B + S - 1) / S;
  if (count) {
    switch (S) {
      case 1: launch_q_S<1, true>(a, st); break;
      case 4: launch_q_S<4, true>(a, st); break;
      case 5: launch_q_S<5, true>(a, st); break;
      case 6: launch_q_S<6, true>(a, st); break;
      case 7: launch_q_S<7, true>(a, st); break;
      case 16: launch_q_S<16, true>(a, st); break;
      default: launch_q_S<8, true>(a, st); break;
    }
  } else {
    switch (S) {
      case 1: launch_q_S<1, false>(a, st); break;
      case 4: launch_q_S<4, false>(a, st); break;
      case 5: launch_q_S<5, false>(a, st); break;
      case 6: launch_q_S<6, false>(a, st); break;
      case 7: launch_q_S<7, false>(a, st); break;
      case 16: launch_q_S<16, false>(a, st); break;
      default: launch_q_S<8, false>(a, st); break;
    }
  }
}

}  // namespace gsr
