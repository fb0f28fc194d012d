// k_backward.cu — backward of stage a4 (SURVEY.md §8(f)-4 follow-on; the objective
// is a function of the rendered images, so its gradient enters through dL/d(image)).
//
// Given g[b] = dL/d(image of state b) for the B states of the frame a forward call has just rendered, the gradient
// of L with respect to the 2-D quantities of every projected record that the compositor read, summed over the
// states and pixels that use the record:
//     grad[record][12] = d/d( rgb[3], rgb with SH residual[3], opacity, A, B, Cq, m_x, m_y )
// Per pixel, with the accepted records i = 1..n in list order (cb = c - bg, w_i = alpha_i T_i):
//     pixel - bg = sum_i w_i cb_i
//     dL/dcb_i    = w_i g
//     dL/dalpha_i = T_i (g . cb_i) - (Gf - G_i) / (1 - alpha_i),  G_i = sum_{j<=i} w_j (g . cb_j),  Gf = g . (pixel - bg)
//     dalpha/do = exp(-q), dalpha/dq = -alpha  (both 0 where the cap 0.99 is active or the cut failed)
//     dq/dA = dx^2, dq/dB = dx dy, dq/dCq = dy^2, dq/dm_x = 2 A dx + B dy, dq/dm_y = B dx + 2 Cq dy
// The suffix of the pixel is taken as (final pixel) - (prefix), so the list is walked front to back exactly like the
// forward pass — same quadrant lists, same staging, same decisions bit for bit (alpha, the cut, the stop rule are
// the forward's operations on the same operands) — and the forward image is an input.
//
// Layout of the work: the forward's (k_composite_q.cu): one warp per 8x8 quadrant x S states, two pixels per lane on
// packed FP32; per (pixel pair, state) T, E = G - Gf and the constants g[3] live in registers (10 per slot).
// Per record the 12 partial sums of the lane's pixels and states are reduced over the warp through shared memory,
// eight records at a time, and added to grad with three vector atomics per record (below).
// Float atomics make the summation order, hence the last bits of grad, run-dependent; parity is by tolerance.
#include "composite_common.cuh"
#include "gsr_internal.h"

namespace gsr {

struct BackwardArgs {
  const float4* rec;
  const uint2* qlist;
  const uint2* qrange;
  const int8_t* depth;   // [B, C]
  int32_t B, C, nsb;
  int32_t W, H, TX, tiles;
  float bg[3];
  const float* images;   // [B,H,W,3] forward output
  const float* gimg;     // [B,H,W,3] dL/d(image)
  float* grad;           // [records, 12]
  uint32_t n_items;        // tiles * 4 * nsb
  uint32_t* work_counter;  // zeroed before the launch
  // tile-level state dedup (k_tile_dedup), or all nullptr: slot = signature class of the tile
  const uint32_t *uorder, *upos, *n_unique;
};

// Reduction of the per-lane partial sums over the warp, through shared memory and kGroup records at a time: every
// lane stores its 12 partials of a record as three float4 (row of 12 floats per lane, record stride kPartStride:
// conflict-free stores and loads); when kGroup records are pending, lane (r = lane % kGroup, h = lane / kGroup < 3)
// adds the h-th float4 of record r over the 32 source lanes and issues ONE vector reduction to grad
// (red.global.add.v4.f32).  Per record: 3 STS.128 + 4 LDS.128-and-add steps per lane instead of a 5-deep shuffle
// butterfly of 16 SHFL + ~45 FSEL / FADD, and 3 vector atomics instead of 12 scalar ones.
#ifndef GSR_BW_GROUP
#define GSR_BW_GROUP 8
#endif
constexpr int kGroup = GSR_BW_GROUP;
constexpr int kSlotGroup = 4;  // slots tested together before the per-slot tests (k_backward_q)
constexpr int kPartStride = 32 * 12 + 4;  // floats; + 4: the kGroup rows of a quarter-warp load fall in distinct banks

__device__ __forceinline__ void sts128f(uint32_t addr, float x, float y, float z, float w) {
  asm volatile("st.shared.v4.f32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "f"(x), "f"(y), "f"(z), "f"(w) : "memory");
}
__device__ __forceinline__ void red_add_v4(float* p, float x, float y, float z, float w) {
  asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(p), "f"(x), "f"(y), "f"(z), "f"(w) : "memory");
}
__device__ __forceinline__ float rcp_approx_ftz(float x) {
  float y;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}

// One state slot, two pixels (header).  T and E = G - Gf (the prefix minus the whole pixel: minus the suffix) are
// carried scaled by 2^40 like the forward's T.
//   dal  += s (T u + E' rinv)               accumulated dL/dalpha of the record over the slots
//   dc*  += (s w) g                          accumulated colour gradient
__device__ __forceinline__ void slot_backward(f32x2& T, f32x2& E, f32x2 gr, f32x2 gg, f32x2 gb, f32x2 alpha2,
                                              f32x2 rinv2, float cr, float cg, float cb, f32x2& dal, f32x2& dcr,
                                              f32x2& dcg, f32x2& dcb) {
  f32x2 u = mul2(gr, pack2(cr, cr));
  u = fma2(gg, pack2(cg, cg), u);
  u = fma2(gb, pack2(cb, cb), u);
  const f32x2 w = mul2(alpha2, T);
  f32x2 Tn;
  asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(Tn) : "l"(T), "l"(w));
  float tl, th;
  unpack2(Tn, tl, th);
  asm("add.rn.sat.f32 %0, %0, 0fCCD1B716;" : "+f"(tl));  // the forward's stop rule: s = [T' >= 1e-4]
  asm("add.rn.sat.f32 %0, %0, 0fCCD1B716;" : "+f"(th));
  const f32x2 s = pack2(tl, th);
  const f32x2 ws = mul2(w, s);
  const f32x2 tu = mul2(T, u);
  E = fma2(ws, u, E);
  const f32x2 t1 = fma2(E, rinv2, tu);  // T u - (Gf - G) / (1 - alpha)
  dal = fma2(s, t1, dal);
  dcr = fma2(ws, gr, dcr);
  dcg = fma2(ws, gg, dcg);
  dcb = fma2(ws, gb, dcb);
  T = Tn;
}

#ifndef GSR_BW_MINB
#define GSR_BW_MINB 12
#endif
template <int S>
__global__ void __launch_bounds__(32, GSR_BW_MINB) k_backward_q(const BackwardArgs a) {
  extern __shared__ uint16_t s_tab[];  // [C][4]: slots (bit s) whose state has depth == 0, >= 1, >= 2, >= 3
  __shared__ __align__(16) float4 s_rec[2][kChunk * 4];
  __shared__ uint32_t s_tag[2][kChunk];  // act | res << 16
  __shared__ uint32_t s_rid[2][kChunk];  // record id (row of grad)
  __shared__ __align__(16) float s_part[kGroup * kPartStride];  // pending per-lane partials: [record][lane][12]
  __shared__ uint32_t s_grid[kGroup];                           // their record ids
  __shared__ int s_rep[S];                 // representative state of slot s, -1 = empty slot
  __shared__ uint32_t s_mlo[S], s_mhi[S];  // members of the class: uorder[tile*B + [mlo, mhi))

  const int lane = threadIdx.x;
  for (;;) {  // persistent warps: work items (tile, quadrant, state block) from a counter, as in k_composite_q
  uint32_t item = 0;
  if (lane == 0) item = atomicAdd(a.work_counter, 1u);
  item = __shfl_sync(0xffffffffu, item, 0);
  if (item >= a.n_items) break;
  const uint32_t tq = item / (uint32_t)a.nsb;  // 4 * tile + quadrant
  const int sb = (int)(item - tq * (uint32_t)a.nsb);
  const int tile = (int)(tq >> 2), quad = (int)(tq & 3u);
  const int b0 = sb * S;  // first slot of this block: a state index, or a class index when dedup is on

  // With tile-level dedup slot s is the s-th signature class of this tile from b0 on.  The members of a class
  // have bitwise identical tile pixels, hence identical T, alpha, w along the list, and the gradient is linear in
  // g: the sum over the members of their gradients is the gradient for the SUM of their g.  One walk per class.
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
  const int x = tx * kTile + 8 * (quad & 1) + (lane & 7);
  const int ya = ty * kTile + 8 * (quad >> 1) + (lane >> 3), yb = ya + 4;
  const bool in_a = x < a.W && ya < a.H, in_b = x < a.W && yb < a.H;
  float px = (float)x + 0.5f;
  f32x2 npy2 = pack2(-((float)ya + 0.5f), -((float)yb + 0.5f));
  asm volatile("" : "+f"(px), "+l"(npy2));
  const uint32_t rec_base = (uint32_t)__cvta_generic_to_shared(&s_rec[0][0]);
  const uint32_t tag_base = (uint32_t)__cvta_generic_to_shared(&s_tag[0][0]);
  const uint32_t rid_base = (uint32_t)__cvta_generic_to_shared(&s_rid[0][0]);
  const uint32_t lt = (1u << lane) - 1u;
  const uint32_t part_base = (uint32_t)__cvta_generic_to_shared(&s_part[0]);
  const uint32_t grid_base = (uint32_t)__cvta_generic_to_shared(&s_grid[0]);
  uint32_t n_pend = 0;  // records waiting in s_part (warp-uniform)
  auto flush = [&](uint32_t n) {
    __syncwarp();
    const uint32_t r = (uint32_t)lane % kGroup, h = (uint32_t)lane / kGroup;
    if (h < 3 && r < n) {
      const uint32_t src = part_base + 4u * (r * kPartStride + 4u * h);
      float4 acc0 = lds128(src), acc1 = lds128(src + 48u);
#pragma unroll
      for (int l = 2; l < 32; l += 2) {
        const float4 t0 = lds128(src + 48u * l), t1 = lds128(src + 48u * (l + 1));
        acc0.x += t0.x; acc0.y += t0.y; acc0.z += t0.z; acc0.w += t0.w;
        acc1.x += t1.x; acc1.y += t1.y; acc1.z += t1.z; acc1.w += t1.w;
      }
      acc0.x += acc1.x; acc0.y += acc1.y; acc0.z += acc1.z; acc0.w += acc1.w;
      if (acc0.x != 0.0f || acc0.y != 0.0f || acc0.z != 0.0f || acc0.w != 0.0f)
        red_add_v4(a.grad + 12 * (size_t)lds32(grid_base + 4u * r) + 4 * h, acc0.x * kInvTScale, acc0.y * kInvTScale,
                   acc0.z * kInvTScale, acc0.w * kInvTScale);
    }
    __syncwarp();
  };

  // per (pixel pair, state): T (scaled by 2^40), E = (prefix of w (g . cb)) - Gf (scaled), and the constants g[3]
  f32x2 T2[S], E2[S], gr2[S], gg2[S], gb2[S];
  const size_t img = (size_t)a.H * a.W * 3;
  const uint32_t* const mem = a.n_unique ? a.uorder + (size_t)tile * a.B : nullptr;
  const size_t po_a = ((size_t)ya * a.W + x) * 3, po_b = ((size_t)yb * a.W + x) * 3;
  {
    // g of a class = the sum of its members' g, in uorder order.  The classes of this block are consecutive in
    // uorder, so the members of all S slots are ONE range [f_lo, f_hi): walked kGBatch members at a time with all
    // their loads in flight together (6 per member and lane; the member indices one batch ahead), the running sum
    // parked in shared memory (s_part, idle until the first record) whenever the walk crosses into the next class.
    static_assert(S * 6 * 32 <= kGroup * kPartStride, "the class sums are parked in s_part");
    constexpr int kGBatch = 8;
    const int n_valid = n_slots - b0 < S ? n_slots - b0 : S;
    const uint32_t f_lo = mem ? s_mlo[0] : (uint32_t)b0, f_hi = mem ? s_mhi[n_valid - 1] : (uint32_t)(b0 + n_valid);
    float acc[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
    int cur = 0;
    uint32_t bound = mem ? s_mhi[0] : f_lo + 1u;
    auto park = [&](int slot) {
#pragma unroll
      for (int c = 0; c < 6; ++c) {
        sts32(part_base + 4u * (uint32_t)((slot * 6 + c) * 32 + lane), __float_as_uint(acc[c]));
        acc[c] = 0.0f;
      }
    };
    uint32_t idx_nxt = 0;
    if (mem && f_lo + (uint32_t)lane < f_hi && lane < kGBatch) idx_nxt = __ldg(mem + f_lo + lane);
    for (uint32_t base = f_lo; base < f_hi; base += kGBatch) {
      const uint32_t idx_cur = idx_nxt;
      if (mem && base + kGBatch + (uint32_t)lane < f_hi && lane < kGBatch) idx_nxt = __ldg(mem + base + kGBatch + lane);
      float v[kGBatch][6];
#pragma unroll
      for (int k = 0; k < kGBatch; ++k) {
        const uint32_t sid = mem ? __shfl_sync(0xffffffffu, idx_cur, k) : base + k;
        const bool have = base + k < f_hi;
        const float* gp = a.gimg + (size_t)sid * img;
#pragma unroll
        for (int ch = 0; ch < 3; ++ch) {
          v[k][ch] = have && in_a ? __ldg(gp + po_a + ch) : 0.0f;
          v[k][3 + ch] = have && in_b ? __ldg(gp + po_b + ch) : 0.0f;
        }
      }
#pragma unroll
      for (int k = 0; k < kGBatch; ++k) {
        if (base + k < f_hi) {
          if (base + k == bound) {  // warp-uniform: classes are non-empty, so one step at most
            park(cur);
            ++cur;
            bound = mem ? s_mhi[cur] : bound + 1u;
          }
#pragma unroll
          for (int c = 0; c < 6; ++c) acc[c] += v[k][c];
        }
      }
    }
    park(cur);
    __syncwarp();
#pragma unroll
    for (int s = 0; s < S; ++s) {
      const int rep = s_rep[s];
      const bool on = rep >= 0;
      float g[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f}, gf[2] = {0.f, 0.f};
      if (on) {
#pragma unroll
        for (int c = 0; c < 6; ++c) g[c] = __uint_as_float(lds32(part_base + 4u * (uint32_t)((s * 6 + c) * 32 + lane)));
        const float* ip = a.images + (size_t)rep * img;
#pragma unroll
        for (int h = 0; h < 2; ++h) {
          if (h ? in_b : in_a) {
            float dot = 0.0f;
#pragma unroll
            for (int ch = 0; ch < 3; ++ch)
              dot = __fmaf_rn(g[3 * h + ch], __fsub_rn(__ldg(ip + (h ? po_b : po_a) + ch), a.bg[ch]), dot);
            gf[h] = dot * kTScale;
          }
        }
      }
      T2[s] = pack2(on && in_a ? kTScale : 0.0f, on && in_b ? kTScale : 0.0f);
      E2[s] = pack2(-gf[0], -gf[1]);
      gr2[s] = pack2(g[0], g[3]); gg2[s] = pack2(g[1], g[4]); gb2[s] = pack2(g[2], g[5]);
    }
    __syncwarp();  // s_part is free again
  }

  const uint2 qr = a.qrange[tq];
  const uint32_t n_ent = qr.y - qr.x;
  const uint2* const list = a.qlist + qr.x;

  auto stage = [&](uint2 e, bool have, int buf) -> uint32_t {
    uint32_t act = 0, res = 0;
    if (have) {
      const uint32_t meta = e.y, cls = meta >> 16;
      const uint16_t* t = s_tab + 4 * (meta & 0xFFFFu);
      if (cls >= 16) {
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
      sts32(rid_base + (uint32_t)buf * (kChunk * 4u) + 4u * pos, e.x);
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
    uint32_t n_nxt = 0;
    if (base + kChunk < n_ent) {
      n_nxt = stage(e_next, base + kChunk + (uint32_t)lane < n_ent, buf ^ 1);
      if (base + 2 * kChunk + (uint32_t)lane < n_ent) e_next = __ldg(list + base + 2 * kChunk + lane);
      cp_async_wait<1>();
    } else {
      cp_async_wait<0>();
    }
    __syncwarp();
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
    const uint32_t ib0 = rid_base + (uint32_t)buf * (kChunk * 4u);
#pragma unroll 1
    for (uint32_t j = 0; j < n_cur; ++j) {
      const uint32_t addr = rb0 + 64u * j;
      const uint32_t tag = lds32(tb0 + 4u * j);
      const uint32_t actl = tag & walive;
      if (actl == 0) continue;
      const float4 h0 = lds128(addr);        // {m_x, m_y, A, B}
      const float4 hq = lds128(addr + 16u);  // {Cq, tau, o, -}
      // the forward's alpha evaluation, operation for operation
      const float dx = __fsub_rn(h0.x, px);
      const f32x2 dy2 = add2(npy2, pack2(h0.y, h0.y));
      const float u = __fmul_rn(h0.z, dx);
      const f32x2 s2 = fma2(dy2, pack2(h0.w, h0.w), pack2(u, u));
      f32x2 q2 = mul2(s2, pack2(dx, dx));
      const f32x2 v2 = mul2(dy2, pack2(hq.x, hq.x));
      q2 = fma2(v2, dy2, q2);
      float qa, qb;
      unpack2(q2, qa, qb);
      const bool pass_a = !(qa > hq.y), pass_b = !(qb > hq.y);
      const float e_a = ex2_approx_ftz(__fmul_rn(qa, -1.4426950408889634f));
      const float e_b = ex2_approx_ftz(__fmul_rn(qb, -1.4426950408889634f));
      const float raw_a = __fmul_rn(hq.z, e_a), raw_b = __fmul_rn(hq.z, e_b);
      const float al_a = pass_a ? fminf(kAlphaCap, raw_a) : 0.0f, al_b = pass_b ? fminf(kAlphaCap, raw_b) : 0.0f;
      // gradients flow through alpha only where the cut passed and the cap is not active
      const float m_a = (pass_a && raw_a <= kAlphaCap) ? 1.0f : 0.0f, m_b = (pass_b && raw_b <= kAlphaCap) ? 1.0f : 0.0f;
      const f32x2 alpha2 = pack2(al_a, al_b);
      const f32x2 rinv2 = pack2(rcp_approx_ftz(1.0f - al_a), rcp_approx_ftz(1.0f - al_b));  // 1 - alpha in [0.01, 1]
      f32x2 dal = pack2(0.f, 0.f);
      f32x2 dc0[3] = {dal, dal, dal}, dc1[3] = {dal, dal, dal};
      const uint32_t act1 = actl & (tag >> 16), act0 = actl ^ act1;
      {
        const float4 k0 = lds128(addr + 32u);  // {rgb - bg, -}
        // the slots are tested four at a time first: a record is present in ~2 of the 12 classes of a block, so most
        // groups are skipped with one test instead of four (measured: 6.67 -> 6.43 ms with both passes grouped)
#pragma unroll
        for (int g4 = 0; g4 < S; g4 += kSlotGroup)
          if (act0 & (((1u << kSlotGroup) - 1u) << g4)) {
#pragma unroll
            for (int s = g4; s < g4 + kSlotGroup && s < S; ++s)
              if ((act0 >> s) & 1u)
                slot_backward(T2[s], E2[s], gr2[s], gg2[s], gb2[s], alpha2, rinv2, k0.x, k0.y, k0.z, dal, dc0[0], dc0[1], dc0[2]);
          }
      }
      if (act1 != 0) {
        const float4 k1 = lds128(addr + 48u);  // {rgb with SH residual - bg, -}
#pragma unroll
        for (int g4 = 0; g4 < S; g4 += kSlotGroup)
          if (act1 & (((1u << kSlotGroup) - 1u) << g4)) {
#pragma unroll
            for (int s = g4; s < g4 + kSlotGroup && s < S; ++s)
              if ((act1 >> s) & 1u)
                slot_backward(T2[s], E2[s], gr2[s], gg2[s], gb2[s], alpha2, rinv2, k1.x, k1.y, k1.z, dal, dc1[0], dc1[1], dc1[2]);
          }
      }
      // per pixel: dL/do = exp(-q) dal, dL/dq = -alpha dal, then the chain through q; the two pixels added
      float v[12];
#pragma unroll
      for (int ch = 0; ch < 3; ++ch) {
        float lo, hi;
        unpack2(dc0[ch], lo, hi); v[ch] = lo + hi;
        unpack2(dc1[ch], lo, hi); v[3 + ch] = lo + hi;
      }
      float da_a, da_b, dya, dyb;
      unpack2(dal, da_a, da_b);
      unpack2(dy2, dya, dyb);
      da_a *= m_a; da_b *= m_b;
      const float dq_a = -al_a * da_a, dq_b = -al_b * da_b;
      v[6] = e_a * da_a + e_b * da_b;
      v[7] = (dq_a + dq_b) * dx * dx;
      v[8] = (dq_a * dya + dq_b * dyb) * dx;
      v[9] = dq_a * dya * dya + dq_b * dyb * dyb;
      v[10] = dq_a * (2.0f * h0.z * dx + h0.w * dya) + dq_b * (2.0f * h0.z * dx + h0.w * dyb);
      v[11] = dq_a * (h0.w * dx + 2.0f * hq.x * dya) + dq_b * (h0.w * dx + 2.0f * hq.x * dyb);
      const uint32_t dst = part_base + 4u * (n_pend * kPartStride + 12u * (uint32_t)lane);
      sts128f(dst, v[0], v[1], v[2], v[3]);
      sts128f(dst + 16u, v[4], v[5], v[6], v[7]);
      sts128f(dst + 32u, v[8], v[9], v[10], v[11]);
      if (lane == 0) sts32(grid_base + 4u * n_pend, lds32(ib0 + 4u * j));
      if (++n_pend == kGroup) {
        flush(kGroup);
        n_pend = 0;
      }
    }
    n_cur = n_nxt;
    __syncwarp();
  }
  if (n_pend) flush(n_pend);
  __syncwarp();  // the shared tables and buffers are rewritten by the next item
  }
}

#ifndef GSR_BW_S
#define GSR_BW_S 12
#endif
constexpr int kBackwardStateBlock = GSR_BW_S;  // measured on cfg1 (ms per 256-state frame): S = 8: 7.6, 9: 7.2, 10: 6.8, 12: 6.67, 14: 11.6

extern thread_local int g_dedup;  // k_composite.cu: option "dedup" of the calling thread

void launch_backward(const DeviceScene& sc, const WsHeader& h, Workspace& ws, const float* images, const float* gimg,
                     float* grad, cudaStream_t st) {
  const int n_rec = sc.N * sc.V;
  if (n_rec > 0) cudaMemsetAsync(grad, 0, sizeof(float) * 12 * (size_t)n_rec, st);
  if (h.B == 0 || n_rec == 0) return;
  // The signature classes are rebuilt here (k_tile_dedup, ~1 % of the pass) rather than taken from the forward
  // call: that call may have run with the option off, or over chunks of a larger batch.
  FrameParams fp{};
  fp.W = h.W; fp.H = h.H; fp.TX = h.TX; fp.TY = h.TY;
  const bool dedup = g_dedup && launch_tile_dedup(sc, fp, ws, ws.depth, h.B, st);
  BackwardArgs a;
  a.rec = ws.rec; a.qlist = ws.qlist; a.qrange = ws.qrange; a.depth = ws.depth;
  a.B = h.B; a.C = sc.C;
  a.nsb = (h.B + kBackwardStateBlock - 1) / kBackwardStateBlock;
  a.W = h.W; a.H = h.H; a.TX = h.TX; a.tiles = h.TX * h.TY;
  a.bg[0] = sc.bg[0]; a.bg[1] = sc.bg[1]; a.bg[2] = sc.bg[2];
  a.images = images; a.gimg = gimg; a.grad = grad;
  a.uorder = dedup ? ws.uorder : nullptr; a.upos = dedup ? ws.upos : nullptr; a.n_unique = dedup ? ws.n_unique : nullptr;
  const size_t smem = sizeof(uint16_t) * 4 * (size_t)sc.C;
  // static (staging + the pending partials, ~17 KB) + dynamic (the presence table, 8 bytes per cluster) passes the
  // default 48 KB from C ~ 3900 on: opt in whenever the sum does
  cudaFuncAttributes fa;
  cudaFuncGetAttributes(&fa, k_backward_q<kBackwardStateBlock>);
  if (smem + fa.sharedSizeBytes > 48 * 1024)
    cudaFuncSetAttribute(k_backward_q<kBackwardStateBlock>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                         (int)(sizeof(uint16_t) * 4 * kMaxC));
  const long long items = (long long)a.tiles * 4 * a.nsb;
  int dev = 0, sms = 1, per_sm = 1;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_backward_q<kBackwardStateBlock>, 32, smem);
  const long long wave = (long long)sms * (per_sm > 0 ? per_sm : 1);
  a.n_items = (uint32_t)items;
  a.work_counter = ws.work_counter;
  cudaMemsetAsync(ws.work_counter, 0, sizeof(uint32_t), st);
  k_backward_q<kBackwardStateBlock><<<(unsigned)(items < wave ? items : wave), 32, smem, st>>>(a);
  count_launches(1);
}

}  // namespace gsr
