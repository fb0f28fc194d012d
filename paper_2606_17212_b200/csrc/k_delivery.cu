// k_delivery.cu — delivery-mask sampler: the step immediately before
// the hot path.  "A training world samples capacity, RTT, display deadline, IID erasure, and a Gilbert-Elliott
// burst process.  Packet dependencies are enforced after delivery, then converted to cluster-layer masks"
// (PAPER.md:64); "A cluster-layer is usable only when all chunks in its dependency closure are usable"
// (PAPER.md:185).  Readings H1-H6: packets of <= 1200 B per completion group, sent group by
// group in a given order; a per-world packet budget stands for capacity / RTT / deadline; IID loss OR a
// two-state Gilbert-Elliott channel; a group is usable iff all its packets arrived; level = closure.
// Randomness is counter-based: Philox4x32-10, key = seed, counter = (packet, world, 0, 0); an event of
// probability p happens iff a 32-bit word is < floor(p * 2^32) — integer decisions, bit-exact by construction.
//
// One warp per world.  The warp takes 32 consecutive packets per iteration; the Gilbert-Elliott chain is
// sequential in the packet index, so each lane turns its transition word into a map {Good,Bad} -> {Good,Bad}
// (2 bits), the maps are composed with a warp inclusive scan (composition is associative), and the carry-in
// state is applied.  Lost packets clear their group's bit in a per-world table in shared memory.
#include "gsr_internal.h"

namespace gsr {

__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0,
                                              uint32_t k1, uint32_t out[4]) {
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    const uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
    const uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
    const uint32_t n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
    c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
    k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

struct LossThresholds {  // floor(p * 2^32) clamped to [0, 2^32], evaluated on the host in double
  unsigned long long iid, gb, bg, e_good, e_bad, pi_bad;
  uint32_t key0, key1;
};

constexpr int kDelWarps = 4;  // worlds per CTA

// pk_start[k] = index of the first packet of the k-th group IN SEND ORDER, pk_start[4C] = total packets
__global__ void k_packet_starts(const long long* __restrict__ raw, const int* __restrict__ order, int n_groups,
                                long long* __restrict__ pk_start, int* __restrict__ err) {
  if (blockIdx.x != 0 || threadIdx.x != 0) return;
  long long acc = 0;
  for (int k = 0; k < n_groups; ++k) {
    pk_start[k] = acc;
    const int g = order[k];
    if ((unsigned)g >= (unsigned)n_groups) {  // not a group id: sends nothing, the caller is told
      if (err) atomicOr(err, kBadOrder);
      continue;
    }
    acc += (raw[g] + 1199) / 1200;
  }
  pk_start[n_groups] = acc;
}

__global__ void __launch_bounds__(32 * kDelWarps) k_sample_delivery(const long long* __restrict__ pk_start,
                                                                    const int* __restrict__ order, int C,
                                                                    LossThresholds th,
                                                                    const int* __restrict__ budget, int W, int world0,
                                                                    uint8_t* __restrict__ mask,
                                                                    int8_t* __restrict__ levels) {
  extern __shared__ uint32_t s_usable[];  // [kDelWarps][ceil(C/8)]: nibble c & 7 of word c >> 3, bit l = group (c, l) still usable
  const int lane = threadIdx.x & 31, wq = threadIdx.x >> 5;
  const int w = blockIdx.x * kDelWarps + wq;
  const int words = (C + 7) >> 3;
  uint32_t* usable = s_usable + (size_t)wq * words;
  for (int k = lane; k < words; k += 32) usable[k] = 0xFFFFFFFFu;
  __syncwarp();
  if (w >= W) return;
  const int n_groups = 4 * C;
  const long long n_packets = pk_start[n_groups];
  const long long my_budget = budget ? (long long)budget[w] : n_packets;
  uint32_t bad = 0;  // carry: channel state after the last packet of the previous iteration
  int gpos = 0;      // send-order position of the group holding this iteration's first packet (monotone)
  for (long long base = 0; base < n_packets; base += 32) {
    const long long i = base + lane;
    const bool have = i < n_packets;
    uint32_t x[4] = {0u, 0u, 0u, 0u};
    if (have) philox4x32_10((uint32_t)i, (uint32_t)(world0 + w), 0u, 0u, th.key0, th.key1, x);
    // transition map of packet i: bit 0 = next state from Good, bit 1 = next state from Bad (1 = Bad)
    uint32_t map = 0x2u;  // identity (lanes past the end)
    if (have) {
      if (i == 0) {
        const uint32_t s0 = (unsigned long long)x[3] < th.pi_bad;  // stationary draw, whatever the carry
        map = s0 | (s0 << 1);
      } else {
        const uint32_t from_good = (unsigned long long)x[1] < th.gb;        // G -> B
        const uint32_t from_bad = !((unsigned long long)x[1] < th.bg);      // B stays B unless B -> G
        map = from_good | (from_bad << 1);
      }
    }
    // inclusive scan of map composition: (later o earlier)(s) = later[earlier[s]]
#pragma unroll
    for (int off = 1; off < 32; off <<= 1) {
      const uint32_t prev = __shfl_up_sync(0xffffffffu, map, off);
      if (lane >= off) {
        const uint32_t g = (map >> (prev & 1u)) & 1u, b = (map >> ((prev >> 1) & 1u)) & 1u;
        map = g | (b << 1);
      }
    }
    const uint32_t state = (map >> bad) & 1u;  // channel state of packet i
    bool arrived = true;
    if (have) {
      const bool lost = (unsigned long long)x[0] < th.iid ||
                        (unsigned long long)x[2] < (state ? th.e_bad : th.e_good);
      arrived = !lost && i < my_budget;
    }
    bad = __shfl_sync(0xffffffffu, state, 31);
    // group of packet i: the last send-order position k with pk_start[k] <= i (empty groups share a start
    // and hold no packet).  Search forward from the iteration's first group.
    while (gpos + 1 < n_groups && pk_start[gpos + 1] <= base) ++gpos;
    if (have && !arrived) {
      int lo = gpos, hi = n_groups - 1;  // largest k in [gpos, n_groups) with pk_start[k] <= i
      while (lo < hi) {
        const int mid = (lo + hi + 1) >> 1;
        if (pk_start[mid] <= i) lo = mid; else hi = mid - 1;
      }
      const int g = order[lo];  // in range: k_packet_starts gives an invalid entry no packet
      if ((unsigned)g < 4u * (unsigned)C)
        atomicAnd(&usable[g >> 5], ~(1u << (g & 31)));  // g = 4c + l: word c >> 3, bit 4 (c & 7) + l
    }
  }
  __syncwarp();
  for (int c = lane; c < C; c += 32) {
    const uint32_t m = (usable[c >> 3] >> (4 * (c & 7))) & 0xFu;
    mask[(size_t)w * C + c] = (uint8_t)m;
    if (levels) levels[(size_t)w * C + c] = (int8_t)(__ffs(~m & 0x1Fu) - 2);  // trailing ones - 1
  }
}

static unsigned long long loss_threshold(double p) {
  double t = floor(p * 4294967296.0);
  if (!(t > 0.0)) return 0ull;
  if (t >= 4294967296.0) return 1ull << 32;
  return (unsigned long long)t;
}

size_t delivery_workspace_bytes(int32_t C) { return sizeof(long long) * (4 * (size_t)C + 1); }

void launch_sample_delivery(const long long* raw, const int32_t* order, int32_t C, const gsr_loss_model& m,
                            const int32_t* budget, int32_t W, int32_t world0, uint8_t* mask, int8_t* levels,
                            long long* pk_start, cudaStream_t st) {
  LossThresholds th;
  th.iid = loss_threshold(m.p_iid);
  th.gb = loss_threshold(m.p_gb);
  th.bg = loss_threshold(m.p_bg);
  th.e_good = loss_threshold(m.e_good);
  th.e_bad = loss_threshold(m.e_bad);
  const double den = m.p_gb + m.p_bg;
  th.pi_bad = den > 0.0 ? loss_threshold(m.p_gb / den) : 0ull;
  th.key0 = (uint32_t)(m.seed & 0xFFFFFFFFull);
  th.key1 = (uint32_t)(m.seed >> 32);
  k_packet_starts<<<1, 32, 0, st>>>(raw, order, 4 * C, pk_start, device_error_word());
  count_launches(1);
  if (W == 0) return;
  const size_t smem = sizeof(uint32_t) * kDelWarps * (size_t)((C + 7) >> 3);
  k_sample_delivery<<<(W + kDelWarps - 1) / kDelWarps, 32 * kDelWarps, smem, st>>>(pk_start, order, C, th, budget, W,
                                                                                 world0, mask, levels);
  count_launches(1);
}

}  // namespace gsr
