// pa_sweep.cuh -- a7/a8: theta checkerboard Metropolis sweeps of every replica + E, M from the final lattice.
// PAPER.md:56 (MCMC equilibration at the new temperature), :126-128 (theta), :62 (observables);
// rule and random keying: DESIGN.md "C3" (reading G20), "C4".
//
// Multispin coding WITHIN a replica, lattice in registers.  Every row is split into its two colour planes,
//   plane c of row y, bit k  <->  site x = 2k + ((y + c) & 1)          (colour (x+y)&1 == c)
// and 32 consecutive active sites of a half-sweep (ordinals q = y*(L/2) + k) share one 32-bit "plane word":
//   L >= 64: a plane word is 32 consecutive k of one row; lane g of the replica's 32 lanes holds rows g*RPL ..
//   L <  64: a plane word is 64/L consecutive rows of L/2 bits each; lane g of the replica's N/64 lanes holds word g.
// The four neighbours of a colour-c site (k,y) are colour 1-c sites: rows y-1, y+1 at bit k, row y at bit k and
// row y at bit k-1 (if (y+c) even) or k+1 (if odd), all modulo L/2.  Rows of neighbouring lanes come by warp shuffle.
// The lattice is read from HBM once and written once per step; nothing else touches memory during the sweeps.
//
// Acceptance (C3/C4, G20): a plane word is exactly one keyed group: its 32 keyed Philox words W_0..W_31 hold,
// in bit column p, the 32-bit uniform of the site at bit p (W_0 = most significant bit).  "u < T" is therefore
// evaluated for the 32 sites of the word AT ONCE by a bit-sliced comparator that walks the words most significant
// bit first: one LOP3 tracks the sites whose bits have all been equal to the threshold's so far, one LOP3 remembers
// the last random bit seen while a site was still undecided.  A site is decided at the first bit that differs
// (probability 1/2 per bit).  Every word gets its first two Philox blocks (8 bits: 255 of 256 sites decided, 88 % of the
// words complete) from the lane that owns it; the words that still have an undecided site -- the stragglers -- are
// COMPACTED across the whole thread block into a shared-memory queue and finished densely, one word per thread, so
// that a straggler costs one lane-block instead of a warp-wide iteration.  Blocks that are never computed cannot
// change a decided site, and a word's result does not depend on which thread finishes it, so the result equals the
// plain definition bit for bit.
//
// What the instruction stream looks like matters more than anything else here: on sm_100a LOP3 (ALU pipe) and
// IMAD.WIDE (FMA-heavy pipe) of one SMSP retire together at one warp instruction per 2 cycles (pipe_probe.cu), so the
// kernel's time is its instruction count.  Hence: three-input logic spelled out as lop3.b32 (NVVM splits it otherwise),
// the comparator specialised on the threshold bits by a uniform branch (2 instead of 3 LOP3 per word and bit), one
// half-sweep body for both colours (the loop must fit the 32 KB instruction-cache level), and a straggler push that
// needs no ballots and no atomics (DESIGN.md 8.2 lists the measured steps and the rejected variants).
#pragma once
#include <cstddef>

#include "pa_common.cuh"

// tuning knobs (defaults are the measured best on B200)
#ifndef PA_SWEEP_THREADS
#define PA_SWEEP_THREADS 128
#endif
#ifndef PA_SWEEP_SMALL_THREADS
#define PA_SWEEP_SMALL_THREADS 128
#endif
#ifndef PA_SWEEP_MINB64
#define PA_SWEEP_MINB64 4
#endif
#ifndef PA_SWEEP_MINB128
#define PA_SWEEP_MINB128 4
#endif
#ifndef PA_SWEEP_RW64
#define PA_SWEEP_RW64 4
#endif
#ifndef PA_SWEEP_RW128
#define PA_SWEEP_RW128 1
#endif
#ifndef PA_SWEEP_CMPG
#define PA_SWEEP_CMPG 8
#endif
#ifndef PA_SWEEP_STAGE1
#define PA_SWEEP_STAGE1 2
#endif

namespace pa {

// threshold bits as all-ones / all-zeros masks, most significant bit first (host-filled kernel argument: the
// LOP3s read them straight from the constant bank)
struct SweepArgs {
  uint32_t a[32];  // a[i] = ~0 iff bit (31 - i) of T4 is set
  uint32_t b[32];  // same for T8
  uint32_t kase[8];  // 2 * (bit of T4) + (bit of T8) for the 8 bits of the mandatory blocks (comparator specialisation)
  int theta;
  int mode;  // 0: inside a step -> buffer cur^1, Rnew replicas, theta sweeps keyed with step ordinal st->step + 1
             // 1: init / set_spins -> buffer cur, R replicas, no sweeps (energies only)
             // 2: as 0, but the lattice of slot i is LOADED from slot parent_of[i] of buffer cur (gather-on-load: the
             //    redistribution copy a6 is fused into the sweep's load) and stored to slot i of buffer cur^1
             // 3: multi-GPU shard -> the exchange has put the new local population (Rnew replicas) into buffer cur; theta
             //    sweeps in place.  The sweeps of every mode are keyed by the GLOBAL slot index (slot0_new + i).
};

__device__ __forceinline__ uint32_t even_bits(uint32_t x) {  // bits 0,2,4,.. -> bits 0..15
  x &= 0x55555555u;
  x = (x | (x >> 1)) & 0x33333333u;
  x = (x | (x >> 2)) & 0x0f0f0f0fu;
  x = (x | (x >> 4)) & 0x00ff00ffu;
  x = (x | (x >> 8)) & 0x0000ffffu;
  return x;
}
__device__ __forceinline__ uint32_t spread_bits(uint32_t x) {  // bits 0..15 -> bits 0,2,4,..
  x &= 0x0000ffffu;
  x = (x | (x << 8)) & 0x00ff00ffu;
  x = (x | (x << 4)) & 0x0f0f0f0fu;
  x = (x | (x << 2)) & 0x33333333u;
  x = (x | (x << 1)) & 0x55555555u;
  return x;
}

// one three-input logic operation, spelled out: NVVM otherwise splits und & ~(u ^ g) into an XOR (or a NOT) and an AND
// that ptxas does not always fuse again.  LUT = f(0xF0, 0xCC, 0xAA) for f(a, b, c).
template <int LUT>
__device__ __forceinline__ uint32_t lop3(uint32_t a, uint32_t b, uint32_t c) {
  uint32_t r;
  asm("lop3.b32 %0, %1, %2, %3, %4;" : "=r"(r) : "r"(a), "r"(b), "r"(c), "n"(LUT));
  return r;
}

// one bit of the MSB-first comparator for 32 sites: u = random bits, A / B = the bit of T4 / T8 (all-ones / all-zeros),
// ge1 = sites that compare against T4 (a == 1; the others against T8)
//   v   <- u where the site is still undecided (so that v ends as the random bit AT the deciding position)
//   und <- und & ~(u ^ X),  X = the site's own threshold bit
__device__ __forceinline__ void cmp_bit(uint32_t& und, uint32_t& v, uint32_t u, uint32_t ge1, uint32_t A, uint32_t B) {
  const uint32_t X = lop3<0xCA>(ge1, A, B);  // ge1 ? A : B
  v = lop3<0xCA>(und, u, v);                 // und ? u : v
  und = lop3<0x90>(und, u, X);               // und & ~(u ^ X)
}
__device__ __forceinline__ void cmp_block(uint32_t& und, uint32_t& v, const uint4& w, uint32_t ge1, const uint32_t* a,
                                          const uint32_t* b) {
  cmp_bit(und, v, w.x, ge1, a[0], b[0]);
  cmp_bit(und, v, w.y, ge1, a[1], b[1]);
  cmp_bit(und, v, w.z, ge1, a[2], b[2]);
  cmp_bit(und, v, w.w, ge1, a[3], b[3]);
}

// The same bit for G words at once, specialised on the pair of threshold bits (warp-uniform: a kernel argument).  X is
// 0, ~0, ge1 or ~ge1, so und <- und & ~(u ^ X) is ONE LOP3 in each of the four cases and the comparator costs 2 instead
// of 3 LOP3 per word and bit; the price is one uniform branch per bit and group.
constexpr int lut_swap_a(int l, int sw) { return sw ? (((l & 0x0F) << 4) | (l >> 4)) : l; }  // LUT of f(~a, b, c)
// FIRST: the very first bit of a half-sweep.  und comes in as ge2 (the sites that are NOT compared: und = ~ge2 is folded
// into the LUTs by swapping their nibbles) and v as "all ones", which makes v' = und ? u : 1 = u | ge2.
template <int G, bool FIRST>
__device__ __forceinline__ void cmp_bit_group(uint32_t kase, uint32_t (&und)[G], uint32_t (&v)[G], const uint32_t (&u)[G],
                                              const uint32_t (&ge1)[G]) {
  constexpr int SW = FIRST ? 1 : 0;
#pragma unroll
  for (int i = 0; i < G; ++i) v[i] = FIRST ? (u[i] | und[i]) : lop3<0xCA>(und[i], u[i], v[i]);  // und ? u : v
  switch (kase) {
    case 0u:  // T4 bit 0, T8 bit 0: X = 0      und & ~u
#pragma unroll
      for (int i = 0; i < G; ++i) und[i] = lop3<lut_swap_a(0x30, SW)>(und[i], u[i], 0u);
      break;
    case 3u:  // 1, 1: X = ~0                   und & u
#pragma unroll
      for (int i = 0; i < G; ++i) und[i] = lop3<lut_swap_a(0xC0, SW)>(und[i], u[i], 0u);
      break;
    case 2u:  // 1, 0: X = ge1                  und & ~(u ^ ge1)
#pragma unroll
      for (int i = 0; i < G; ++i) und[i] = lop3<lut_swap_a(0x90, SW)>(und[i], u[i], ge1[i]);
      break;
    default:  // 0, 1: X = ~ge1                 und & (u ^ ge1)
#pragma unroll
      for (int i = 0; i < G; ++i) und[i] = lop3<lut_swap_a(0x60, SW)>(und[i], u[i], ge1[i]);
      break;
  }
}

// ---------------------------------------------------------------------------------------------------
// Straggler queue of one thread block (shared memory).  An item is one plane word that still has undecided sites
// after its two mandatory Philox blocks: the comparator state (und, v), the word's a >= 1 mask, and where its keyed
// words come from (replica slot relative to the block's first slot, first Philox call of the group).
// Protocol per half-sweep h (parity = h & 1), two block barriers:
//   push (owners)  --A--  finish items densely, one per thread; thread 0 clears the OTHER parity's counter  --B--
//   owners OR the late flips of their pushed words into their flip masks.
// Items and results live in separate arrays, so a fast warp that already pushes for h + 1 never touches what a slow
// warp still reads for h; only the counter is double buffered.  A push past CAP (cannot happen for L <= 64, where CAP
// covers every word of the block; 50 sigma away for L = 128) is finished in place by its owner.
// ---------------------------------------------------------------------------------------------------
template <int CAP>
struct SweepQueue {
  uint4 item[CAP];    // und, v, ge1, (slot - slot_base) << 16 | call0
  uint32_t res[CAP];  // late flips of the item
  uint32_t count[2];
  uint32_t pad_[2];   // sizeof is a multiple of 16: queues can be laid side by side
  uint32_t wcount[2][4];  // region form (4 warps, CAP = every word of the block): items of warp w per half-sweep parity
  static constexpr uint32_t OFF_RES = 16u * CAP, OFF_COUNT = 20u * CAP;  // byte offsets (checked in k_sweep*)
  static constexpr uint32_t OFF_WCOUNT = OFF_COUNT + 16u;
};
// REGION form of the queue (4 warps, CAP = every word of the block): per-warp regions, no atomics.  OWNER form on top of
// it (a multiple of 4 words per thread): items name their owner and the late flips come back through per-thread slots.
template <int NW, int THREADS, int CAP>
struct QueueForm {
  static constexpr bool REGION = THREADS == 128 && CAP == NW * THREADS;
  static constexpr bool OWNER = REGION && NW % 4 == 0;
};

// The queue is addressed through its 32-bit shared-window address (taken once per kernel) so that every access is a
// plain LDS / STS / ATOMS with an immediate offset.
__device__ __forceinline__ void sts128(uint32_t addr, uint32_t a, uint32_t b, uint32_t c, uint32_t d) {
  asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "r"(a), "r"(b), "r"(c), "r"(d) : "memory");
}
__device__ __forceinline__ uint4 lds128(uint32_t addr) {
  uint4 r;
  asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "r"(addr) : "memory");
  return r;
}
__device__ __forceinline__ void sts32(uint32_t addr, uint32_t a) {
  asm volatile("st.shared.u32 [%0], %1;" ::"r"(addr), "r"(a) : "memory");
}
__device__ __forceinline__ uint32_t lds32(uint32_t addr) {
  uint32_t r;
  asm volatile("ld.shared.u32 %0, [%1];" : "=r"(r) : "r"(addr) : "memory");
  return r;
}
__device__ __forceinline__ uint32_t atoms_add(uint32_t addr, uint32_t a) {
  uint32_t r;
  asm volatile("atom.shared.add.u32 %0, [%1], %2;" : "=r"(r) : "r"(addr), "r"(a) : "memory");
  return r;
}

// blocks 2..7 of one word: returns the sites of und0 that end with u < T.  The first PA_SWEEP_STAGE2 blocks are computed
// unconditionally and side by side (two independent Philox chains; the thresholds are compile-time offsets): one item
// in 14 needs the second of them, but a warp of 30 items almost always has such an item, and a warp-wide loop iteration
// per extra block costs every lane of the warp a full, latency-bound Philox chain.  A block that is not needed cannot
// change a decided site.  What is still undecided after 16 bits (one item in 4000) goes through the loop.
#ifndef PA_SWEEP_STAGE2
#define PA_SWEEP_STAGE2 1
#endif
__device__ __forceinline__ uint32_t finish_word(uint32_t und, uint32_t v, uint32_t ge1, uint32_t slot, uint32_t call0,
                                                uint32_t c2, uint32_t c3, const PhiloxKey& key, const SweepArgs& sa) {
  const uint32_t und0 = und;
  {
    uint4 w[PA_SWEEP_STAGE2 > 0 ? PA_SWEEP_STAGE2 : 1];
#pragma unroll
    for (int k = 0; k < PA_SWEEP_STAGE2; ++k) w[k] = philox4x32_10(slot, call0 + (uint32_t)(PA_SWEEP_STAGE1 + k), c2, c3, key);
#pragma unroll
    for (int k = 0; k < PA_SWEEP_STAGE2; ++k)
      cmp_block(und, v, w[k], ge1, sa.a + 4 * (PA_SWEEP_STAGE1 + k), sa.b + 4 * (PA_SWEEP_STAGE1 + k));
  }
#pragma unroll 1
  for (uint32_t c = (uint32_t)(PA_SWEEP_STAGE1 + PA_SWEEP_STAGE2); und != 0u; ++c) {
    const uint4 w = philox4x32_10(slot, call0 + c, c2, c3, key);
    cmp_block(und, v, w, ge1, sa.a + 4u * c, sa.b + 4u * c);
    if (c == 7u) {  // all 32 bits equal: u == T is not less
      v |= und;
      und = 0u;
    }
  }
  return ~v & und0;
}

// flip masks of the NW plane words of a lane.  ge1 / ge2: sites with a >= 1 / a >= 2 anti-aligned neighbours;
// call0 = 8 * group.   a >= 2: always flip;  a == 1: flip iff u < T4;  a == 0: flip iff u < T8
// (u < T  <=>  at the first differing bit, most significant first, u has 0).
// Three phases around the two synchronisation points A and B of the queue protocol:
//   accept_phase1    two mandatory Philox blocks per word; stragglers pushed; flip = the sites decided so far   --A--
//   accept_process   the block finishes the queued items densely, one per thread                                 --B--
//   accept_readback  owners OR the late flips of their pushed words into their flip masks
template <int NW, int THREADS, int CAP>
__device__ __forceinline__ void accept_phase1(uint32_t q /* shared address of the SweepQueue<CAP> */, unsigned parity,
                                              const uint32_t (&ge1)[NW], const uint32_t (&ge2)[NW],
                                              const uint32_t (&slot)[NW],  // replica of each word
                                              uint32_t slot_base,          // first slot of the thread block
                                              const uint32_t (&call0)[NW], uint32_t c2, uint32_t c3, const PhiloxKey& key,
                                              const SweepArgs& sa, uint32_t (&flip)[NW], uint32_t (&und)[NW],
                                              unsigned (&idx)[NW]) {
  constexpr unsigned FULL = 0xffffffffu;
  constexpr bool CAN_OVERFLOW = CAP < NW * THREADS;
  uint32_t v[NW];
#pragma unroll
  for (int i = 0; i < NW; ++i) {
    und[i] = ~ge2[i];
    v[i] = 0xffffffffu;
  }
  if constexpr (PA_SWEEP_CMPG > 0 && NW >= PA_SWEEP_CMPG && NW % (PA_SWEEP_CMPG > 0 ? PA_SWEEP_CMPG : 1) == 0) {
    // comparator specialised on the threshold bits, G words per uniform branch (cmp_bit_group)
    constexpr int G = PA_SWEEP_CMPG > 0 ? PA_SWEEP_CMPG : 1;
#pragma unroll
    for (int g0 = 0; g0 < NW; g0 += G) {
      uint32_t gu[G], gv[G], gg[G];
#pragma unroll
      for (int i = 0; i < G; ++i) { gu[i] = ge2[g0 + i]; gv[i] = 0u; gg[i] = ge1[g0 + i]; }  // first bit: FIRST form
#pragma unroll
      for (int c = 0; c < PA_SWEEP_STAGE1; ++c) {
        uint4 w[G];
#pragma unroll
        for (int i = 0; i < G; ++i) w[i] = philox4x32_10(slot[g0 + i], call0[g0 + i] + (uint32_t)c, c2, c3, key);
        uint32_t u[G];
#pragma unroll
        for (int i = 0; i < G; ++i) u[i] = w[i].x;
        if (c == 0) cmp_bit_group<G, true>(sa.kase[0], gu, gv, u, gg);
        else cmp_bit_group<G, false>(sa.kase[4 * c], gu, gv, u, gg);
#pragma unroll
        for (int i = 0; i < G; ++i) u[i] = w[i].y;
        cmp_bit_group<G, false>(sa.kase[4 * c + 1], gu, gv, u, gg);
#pragma unroll
        for (int i = 0; i < G; ++i) u[i] = w[i].z;
        cmp_bit_group<G, false>(sa.kase[4 * c + 2], gu, gv, u, gg);
#pragma unroll
        for (int i = 0; i < G; ++i) u[i] = w[i].w;
        cmp_bit_group<G, false>(sa.kase[4 * c + 3], gu, gv, u, gg);
      }
#pragma unroll
      for (int i = 0; i < G; ++i) { und[g0 + i] = gu[i]; v[g0 + i] = gv[i]; }
    }
  } else {  // few words per lane (L < 64): the branch per bit would cost more than the LOP3 it saves
#pragma unroll
    for (int c = 0; c < PA_SWEEP_STAGE1; ++c) {
#pragma unroll
      for (int i = 0; i < NW; ++i) {
        const uint4 w = philox4x32_10(slot[i], call0[i] + (uint32_t)c, c2, c3, key);
        cmp_block(und[i], v[i], w, ge1[i], sa.a + 4 * c, sa.b + 4 * c);
      }
    }
  }
  const unsigned lane = threadIdx.x & 31u;
  if constexpr (QueueForm<NW, THREADS, CAP>::REGION) {
    // ---- push, region form: warp w owns slots [w * 32 NW, (w + 1) * 32 NW); a lane numbers its own stragglers, one
    // warp-wide exclusive scan of the lanes' counts places them; no ballots, no atomic, no counter to reset ----
    unsigned k = 0u;
#pragma unroll
    for (int i = 0; i < NW; ++i) {
      idx[i] = k;
      k += und[i] != 0u ? 1u : 0u;
    }
    unsigned incl = k;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const unsigned t = __shfl_up_sync(FULL, incl, o);
      if (lane >= (unsigned)o) incl += t;
    }
    const unsigned warp = threadIdx.x >> 5;
    if (lane == 31u) sts32(q + SweepQueue<CAP>::OFF_WCOUNT + 16u * parity + 4u * warp, incl);
    const unsigned first = warp * (unsigned)(32 * NW) + incl - k;
#pragma unroll
    for (int i = 0; i < NW; ++i) {
      idx[i] += first;
      flip[i] = lop3<0x51>(ge2[i], v[i], und[i]);  // (ge2 | ~v) & ~und: the sites decided so far; the rest comes back through q.res
      // the item names its OWNER (thread, word): the dense pass derives the replica from it and writes the late flips
      // into the owner's own result slot
      const uint32_t who = NW % 4 == 0 ? threadIdx.x * (unsigned)NW + (unsigned)i : slot[i] - slot_base;
      if (und[i] != 0u) sts128(q + 16u * idx[i], und[i], v[i], ge1[i], (who << 16) | call0[i]);
    }
  } else {
    // ---- push the stragglers: one shared-memory atomic per warp ----
    const unsigned lt = (1u << lane) - 1u;
    unsigned tot = 0u;
#pragma unroll
    for (int i = 0; i < NW; ++i) {
      const unsigned bal = __ballot_sync(FULL, und[i] != 0u);
      idx[i] = tot + (unsigned)__popc(bal & lt);
      tot += (unsigned)__popc(bal);
    }
    unsigned base = 0u;
    if (tot != 0u) {  // warp-uniform
      if (lane == 0u) base = atoms_add(q + SweepQueue<CAP>::OFF_COUNT + 4u * parity, tot);
      base = __shfl_sync(FULL, base, 0);
    }
#pragma unroll
    for (int i = 0; i < NW; ++i) {
      idx[i] += base;
      flip[i] = lop3<0x51>(ge2[i], v[i], und[i]);  // (ge2 | ~v) & ~und: the sites decided so far; the rest comes back through q.res
      if (CAN_OVERFLOW && und[i] != 0u && idx[i] >= (unsigned)CAP) {  // queue full: the owner finishes its word in place
        flip[i] |= finish_word(und[i], v[i], ge1[i], slot[i], call0[i], c2, c3, key, sa);
        und[i] = 0u;
      }
      if (und[i] != 0u) sts128(q + 16u * idx[i], und[i], v[i], ge1[i], ((slot[i] - slot_base) << 16) | call0[i]);
    }
  }
}

template <int NW, int THREADS, int CAP, class SlotOf>
__device__ __forceinline__ void accept_process(uint32_t q, unsigned parity, uint32_t slot_base, uint32_t c2, uint32_t c3,
                                               const PhiloxKey& key, const SweepArgs& sa) {
  if constexpr (QueueForm<NW, THREADS, CAP>::REGION) {  // region form: the 4 warps' items, densely numbered
    const uint4 cn = lds128(q + SweepQueue<CAP>::OFF_WCOUNT + 16u * parity);
    const unsigned n = cn.x + cn.y + cn.z + cn.w;
    for (unsigned it = threadIdx.x; it < n; it += THREADS) {
      unsigned loc = it, reg = 0u;
      if (loc >= cn.x) {
        loc -= cn.x; reg = 1u;
        if (loc >= cn.y) {
          loc -= cn.y; reg = 2u;
          if (loc >= cn.z) { loc -= cn.z; reg = 3u; }
        }
      }
      const unsigned pos = reg * (unsigned)(32 * NW) + loc;
      const uint4 m = lds128(q + 16u * pos);
      if constexpr (QueueForm<NW, THREADS, CAP>::OWNER) {
        const unsigned owner = m.w >> 16, ot = owner / (unsigned)NW, oi = owner % (unsigned)NW;  // thread and word of the owner
        // result slots: word oi of thread ot lives in 16-byte vector (oi / 4) * THREADS + ot, so that an owner reads its
        // NW results with NW / 4 conflict-free 128-bit loads
        sts32(q + SweepQueue<CAP>::OFF_RES + 16u * ((oi >> 2) * (unsigned)THREADS + ot) + 4u * (oi & 3u),
              finish_word(m.x, m.y, m.z, slot_base + SlotOf::rel(ot, oi), m.w & 0xffffu, c2, c3, key, sa));
      } else {
        sts32(q + SweepQueue<CAP>::OFF_RES + 4u * pos,
              finish_word(m.x, m.y, m.z, slot_base + (m.w >> 16), m.w & 0xffffu, c2, c3, key, sa));
      }
    }
  } else {
    constexpr bool CAN_OVERFLOW = CAP < NW * THREADS;
    unsigned n = lds32(q + SweepQueue<CAP>::OFF_COUNT + 4u * parity);
    if (CAN_OVERFLOW && n > (unsigned)CAP) n = (unsigned)CAP;
    if (threadIdx.x == 0) sts32(q + SweepQueue<CAP>::OFF_COUNT + 4u * (parity ^ 1u), 0u);  // last read before B of the previous half-sweep
    for (unsigned it = threadIdx.x; it < n; it += THREADS) {
      const uint4 m = lds128(q + 16u * it);
      sts32(q + SweepQueue<CAP>::OFF_RES + 4u * it,
            finish_word(m.x, m.y, m.z, slot_base + (m.w >> 16), m.w & 0xffffu, c2, c3, key, sa));
    }
  }
}

// owner form: every thread's result slots start out empty
template <int NW, int THREADS, int CAP>
__device__ __forceinline__ void queue_clear_results(uint32_t q) {
  if constexpr (QueueForm<NW, THREADS, CAP>::OWNER) {
#pragma unroll
    for (int h = 0; h < NW / 4; ++h) sts128(q + SweepQueue<CAP>::OFF_RES + 16u * ((unsigned)h * (unsigned)THREADS + threadIdx.x), 0u, 0u, 0u, 0u);
  }
}

template <int NW, int THREADS, int CAP>
__device__ __forceinline__ void accept_readback(uint32_t q, const uint32_t (&und)[NW], const unsigned (&idx)[NW],
                                                uint32_t (&flip)[NW]) {
  if constexpr (QueueForm<NW, THREADS, CAP>::OWNER) {
    // owner form: the thread's own NW result words (zero unless a pushed word came back), NW / 4 vector loads, and the
    // slots are cleared for the next half-sweep (whose dense pass writes them only after the next barrier A)
    static_assert(NW % 4 == 0, "result slots are 128-bit vectors");
#pragma unroll
    for (int h = 0; h < NW / 4; ++h) {
      const uint32_t a = q + SweepQueue<CAP>::OFF_RES + 16u * ((unsigned)h * (unsigned)THREADS + threadIdx.x);
      const uint4 r = lds128(a);
      flip[4 * h] |= r.x; flip[4 * h + 1] |= r.y; flip[4 * h + 2] |= r.z; flip[4 * h + 3] |= r.w;
      sts128(a, 0u, 0u, 0u, 0u);
    }
  } else {
#pragma unroll
    for (int i = 0; i < NW; ++i)
      if (und[i] != 0u) flip[i] |= lds32(q + SweepQueue<CAP>::OFF_RES + 4u * idx[i]);
  }
}

// the three phases with block barriers at A and B.  Must be called by EVERY thread of the block; lanes without work
// pass ge2 = ~0.
template <int NW, int THREADS, int CAP, class SlotOf>
__device__ __forceinline__ void queued_accept(uint32_t q, unsigned parity, const uint32_t (&ge1)[NW],
                                              const uint32_t (&ge2)[NW], const uint32_t (&slot)[NW], uint32_t slot_base,
                                              const uint32_t (&call0)[NW], uint32_t c2, uint32_t c3, const PhiloxKey& key,
                                              const SweepArgs& sa, uint32_t (&flip)[NW]) {
  uint32_t und[NW];
  unsigned idx[NW];
  accept_phase1<NW, THREADS, CAP>(q, parity, ge1, ge2, slot, slot_base, call0, c2, c3, key, sa, flip, und, idx);
  __syncthreads();  // A: every push of this half-sweep is visible
  accept_process<NW, THREADS, CAP, SlotOf>(q, parity, slot_base, c2, c3, key, sa);
  __syncthreads();  // B: every result is visible
  accept_readback<NW, THREADS, CAP>(q, und, idx, flip);
}

// masks of the sites with a >= 1 and a >= 2 anti-aligned neighbours, straight from the five words (7 LOP3): the four
// neighbours in two pairs, "one of the pair differs from tt" and "both differ"
__device__ __forceinline__ void neighbour_classes(uint32_t tt, uint32_t U, uint32_t D, uint32_t Sm, uint32_t B,
                                                  uint32_t& ge1, uint32_t& ge2) {
  const uint32_t any_ud = lop3<0x7E>(tt, U, D), both_ud = lop3<0x18>(tt, U, D);    // (tt^U)|(tt^D), (tt^U)&(tt^D)
  const uint32_t any_sb = lop3<0x7E>(tt, Sm, B), both_sb = lop3<0x18>(tt, Sm, B);
  ge1 = any_ud | any_sb;
  ge2 = lop3<0xFE>(both_ud, both_sb, any_ud & any_sb);
}

// Second Hamiltonian (D1: 2D +-J spin glass, H = -sum J_ij sigma_i sigma_j): a bond is unsatisfied iff the spins
// differ XOR the coupling is negative.  The host tabulates, for every colour C and every plane word (= keyed group) of a
// half-sweep, which of the four bonds of each active site are negative: bond_mask[C * N/64 + group] = {up, down, same-bit
// neighbour of the row, shifted neighbour of the row}, bit p = site ordinal p of the group.  With the masks XORed into the
// four difference words "a" counts unsatisfied bonds and everything downstream (classes, thresholds, E = 2u - 2N) is
// unchanged.  SG = false compiles the masks away (ferromagnet, eq. 6).
template <bool SG>
__device__ __forceinline__ void neighbour_classes_j(uint32_t tt, uint32_t U, uint32_t D, uint32_t Sm, uint32_t B,
                                                    const uint4& mk, uint32_t& ge1, uint32_t& ge2) {
  if constexpr (SG) {
    const uint32_t d0 = lop3<0x96>(tt, U, mk.x), d1 = lop3<0x96>(tt, D, mk.y), d2 = lop3<0x96>(tt, Sm, mk.z),
                   d3 = lop3<0x96>(tt, B, mk.w);                      // unsatisfied bonds: spins differ XOR negative coupling
    const uint32_t maj = lop3<0xE8>(d0, d1, d2), any3 = lop3<0xFE>(d0, d1, d2);
    ge2 = lop3<0xF8>(maj, any3, d3);                                  // maj | (any3 & d3)
    ge1 = any3 | d3;
  } else {
    neighbour_classes(tt, U, D, Sm, B, ge1, ge2);
  }
}

constexpr int SWEEP_THREADS = PA_SWEEP_THREADS;              // k_sweep (L >= 64)
constexpr int SWEEP_SMALL_THREADS = PA_SWEEP_SMALL_THREADS;  // k_sweep_small (L < 64)

// =====================================================================================================
// L >= 64: a warp holds RW consecutive replicas (lane g holds rows g*RPL .. of each), so that a lane owns
// NWL = RW * RPL * WPP plane words per half-sweep and the block's straggler queue is fed by 8 words per lane.
// =====================================================================================================
template <int L>
struct Geo {
  static constexpr int N = L * L;
  static constexpr int G = 32;                    // lanes per replica
  static constexpr int RPL = L / G;               // rows per lane
  static constexpr int HB = L / 2;                // bits per row per colour plane
  static constexpr int WPP = HB / 32;             // words per row plane
  static constexpr int WR = L / 32;               // raw words per row
  static constexpr int WREP = N / 32;             // words per replica
  static constexpr int RW = L >= 128 ? PA_SWEEP_RW128 : PA_SWEEP_RW64;  // replicas per warp
  static constexpr int NWR = RPL * WPP;           // plane words of one replica per lane and half-sweep
  static constexpr int NWL = RW * NWR;            // plane words per lane and half-sweep
  static constexpr int RPB = (SWEEP_THREADS / 32) * RW;  // replicas per block
};

// replica (relative to the block's first) that word w of thread t belongs to: what the dense pass needs to key an item
template <int L>
struct BigSlotOf {
  static __device__ __forceinline__ uint32_t rel(unsigned t, unsigned w) { return (t >> 5) * (unsigned)Geo<L>::RW + w / (unsigned)Geo<L>::NWR; }
};

// capacity of the block's straggler queue: every word of a half-sweep up to 1024 items, 1024 beyond
template <int NW, int THREADS = SWEEP_THREADS>
struct SweepCap {
  static constexpr int WORDS = NW * THREADS;  // plane words per block and half-sweep
  static constexpr int CAP = WORDS <= 1024 ? WORDS : 1024;
};

template <int L>
struct Lattice {
  using G_ = Geo<L>;
  uint32_t p[2][G_::RPL][G_::WPP];  // colour planes
};

// rotate plane row so that result bit k = source bit k-1 (dir = 0) or k+1 (dir = 1), modulo HB
template <int L>
__device__ __forceinline__ void rot_row(const uint32_t (&s)[Geo<L>::WPP], int dir, uint32_t (&out)[Geo<L>::WPP]) {
  using G_ = Geo<L>;
#pragma unroll
  for (int i = 0; i < G_::WPP; ++i) {
    const uint32_t prev = s[(i + G_::WPP - 1) % G_::WPP], next = s[(i + 1) % G_::WPP];
    const uint32_t left = __funnelshift_l(prev, s[i], 1);   // (s[i] << 1) | (prev >> 31)
    const uint32_t right = __funnelshift_r(s[i], next, 1);  // (s[i] >> 1) | (next << 31)
    out[i] = dir ? right : left;
  }
}

// One half-sweep of the lane's rows of the warp's RW replicas, with the colour as a RUN-TIME value and ONE body for both
// colours: the plane that is updated is always p[0] and the other one p[1]; after the update the two planes trade places (p[1] <- p[0] ^ flip, p[0] <- old
// p[1]), so an even number of half-sweeps leaves them where they were.  Unrolling the two colours instead doubles the
// loop body to 36 KB, which no longer fits the 32 KB instruction cache level an SM's warps share (the guide's I-cache
// table: +5 % steady past 32 KB; ncu: 0.25 no-instruction stalls per issue); one body is 18 KB.  Cost: 16 register moves
// per half-sweep and a run-time rotate amount.  Needs an even number of rows per lane (row parity = r parity).
template <int L, bool SG>
__device__ __forceinline__ void half_sweep_rt(Lattice<L> (&lat)[Geo<L>::RW], uint32_t q, int g, uint32_t C,
                                              uint32_t slot0, uint32_t slot_base, uint32_t c2, uint32_t c3,
                                              const PhiloxKey& key, const SweepArgs& sa,
                                              const uint4* __restrict__ bond_mask) {
  using G_ = Geo<L>;
  static_assert(G_::RPL % 2 == 0, "row parity must not depend on the lane");
  constexpr unsigned FULL = 0xffffffffu;
  constexpr int NWL = G_::NWL;
  const int gu = (g + G_::G - 1) % G_::G, gd = (g + 1) % G_::G;
  const uint32_t sh_even = C ? 31u : 1u, sh_odd = C ? 1u : 31u;  // rotate-left amounts: bit k <- bit k-1 (1) or k+1 (31)
  const uint4* __restrict__ bm = bond_mask + C * (G_::N / 64) + g * G_::RPL * G_::WPP;
  uint32_t ge1[NWL], ge2[NWL], call0[NWL], slots[NWL];
#pragma unroll
  for (int rep = 0; rep < G_::RW; ++rep) {
    uint32_t(&T)[G_::RPL][G_::WPP] = lat[rep].p[0];
    uint32_t(&S)[G_::RPL][G_::WPP] = lat[rep].p[1];
    uint32_t up[G_::WPP], dn[G_::WPP];
#pragma unroll
    for (int i = 0; i < G_::WPP; ++i) {
      up[i] = __shfl_sync(FULL, S[G_::RPL - 1][i], gu, G_::G);
      dn[i] = __shfl_sync(FULL, S[0][i], gd, G_::G);
    }
#pragma unroll
    for (int r = 0; r < G_::RPL; ++r) {
      const uint32_t sh = (r & 1) ? sh_odd : sh_even;  // row y = g * RPL + r uses bit k-1 when (y + C) is even
      uint32_t B[G_::WPP];
      if constexpr (G_::WPP == 1) {
        B[0] = __funnelshift_l(S[r][0], S[r][0], sh);
      } else {
#pragma unroll
        for (int i = 0; i < G_::WPP; ++i) {
          const uint32_t prev = S[r][(i + G_::WPP - 1) % G_::WPP], next = S[r][(i + 1) % G_::WPP];
          const uint32_t left = __funnelshift_l(prev, S[r][i], 1), right = __funnelshift_r(S[r][i], next, 1);
          B[i] = sh == 1u ? left : right;
        }
      }
#pragma unroll
      for (int i = 0; i < G_::WPP; ++i) {
        const int w = rep * G_::NWR + r * G_::WPP + i;
        const uint32_t U = (r > 0) ? S[r > 0 ? r - 1 : 0][i] : up[i];
        const uint32_t D = (r < G_::RPL - 1) ? S[r < G_::RPL - 1 ? r + 1 : 0][i] : dn[i];
        uint4 mk = make_uint4(0u, 0u, 0u, 0u);
        if constexpr (SG) mk = __ldg(bm + r * G_::WPP + i);
        neighbour_classes_j<SG>(T[r][i], U, D, S[r][i], B[i], mk, ge1[w], ge2[w]);
        call0[w] = 8u * ((uint32_t)(g * G_::RPL + r) * G_::WPP + (uint32_t)i);  // group = y * WPP + i
        slots[w] = slot0 + (uint32_t)rep;
      }
    }
  }
  uint32_t flip[NWL];
  queued_accept<NWL, SWEEP_THREADS, SweepCap<NWL>::CAP, BigSlotOf<L>>(q, C, ge1, ge2, slots, slot_base, call0, c2, c3, key, sa, flip);
#pragma unroll
  for (int rep = 0; rep < G_::RW; ++rep)
#pragma unroll
    for (int w = 0; w < G_::NWR; ++w) {
      uint32_t& a = lat[rep].p[0][w / G_::WPP][w % G_::WPP];
      uint32_t& b = lat[rep].p[1][w / G_::WPP][w % G_::WPP];
      const uint32_t updated = a ^ flip[rep * G_::NWR + w];
      a = b;
      b = updated;
    }
}

// number of anti-aligned bonds u (each bond has exactly one colour-0 end) and number of up spins
template <int L, bool SG>
__device__ __forceinline__ void count_bonds(const Lattice<L>& lat, int g, const uint4* __restrict__ bond_mask, int& unsat,
                                            int& ups) {
  using G_ = Geo<L>;
  constexpr unsigned FULL = 0xffffffffu;
  const uint32_t(&T)[G_::RPL][G_::WPP] = lat.p[0];
  const uint32_t(&S)[G_::RPL][G_::WPP] = lat.p[1];
  uint32_t up[G_::WPP], dn[G_::WPP];
  const int gu = (g + G_::G - 1) % G_::G, gd = (g + 1) % G_::G;
#pragma unroll
  for (int i = 0; i < G_::WPP; ++i) {
    up[i] = __shfl_sync(FULL, S[G_::RPL - 1][i], gu, G_::G);
    dn[i] = __shfl_sync(FULL, S[0][i], gd, G_::G);
  }
  int u = 0, pc = 0;
#pragma unroll
  for (int r = 0; r < G_::RPL; ++r) {
    const int y = g * G_::RPL + r;
    uint32_t B[G_::WPP];
    rot_row<L>(S[r], y & 1, B);
#pragma unroll
    for (int i = 0; i < G_::WPP; ++i) {
      const uint32_t U = (r > 0) ? S[r > 0 ? r - 1 : 0][i] : up[i];
      const uint32_t D = (r < G_::RPL - 1) ? S[r < G_::RPL - 1 ? r + 1 : 0][i] : dn[i];
      const uint32_t tt = T[r][i];
      uint4 mk = make_uint4(0u, 0u, 0u, 0u);
      if constexpr (SG) mk = __ldg(bond_mask + y * G_::WPP + i);  // colour 0
      u += __popc(tt ^ U ^ mk.x) + __popc(tt ^ D ^ mk.y) + __popc(tt ^ S[r][i] ^ mk.z) + __popc(tt ^ B[i] ^ mk.w);
      pc += __popc(tt) + __popc(S[r][i]);
    }
  }
  unsat = u;
  ups = pc;
}

// raw row bits (x = 0..L-1 in WR words) <-> colour planes
template <int L>
__device__ __forceinline__ void row_to_planes(const uint32_t (&raw)[Geo<L>::WR], int y_odd,
                                              uint32_t (&p0)[Geo<L>::WPP], uint32_t (&p1)[Geo<L>::WPP]) {
  using G_ = Geo<L>;
#pragma unroll
  for (int i = 0; i < G_::WPP; ++i) {  // even row: colour 0 sits at even x; odd row: at odd x
    const uint32_t ev = even_bits(raw[2 * i]) | (even_bits(raw[2 * i + 1]) << 16);
    const uint32_t od = even_bits(raw[2 * i] >> 1) | (even_bits(raw[2 * i + 1] >> 1) << 16);
    p0[i] = y_odd ? od : ev;
    p1[i] = y_odd ? ev : od;
  }
}
template <int L>
__device__ __forceinline__ void planes_to_row(const uint32_t (&p0)[Geo<L>::WPP], const uint32_t (&p1)[Geo<L>::WPP],
                                              int y_odd, uint32_t (&raw)[Geo<L>::WR]) {
  using G_ = Geo<L>;
#pragma unroll
  for (int i = 0; i < G_::WPP; ++i) {
    const uint32_t ev = y_odd ? p1[i] : p0[i], od = y_odd ? p0[i] : p1[i];
    raw[2 * i] = spread_bits(ev) | (spread_bits(od) << 1);
    raw[2 * i + 1] = spread_bits(ev >> 16) | (spread_bits(od >> 16) << 1);
  }
}

template <int L, bool SG>
__global__ void __launch_bounds__(SWEEP_THREADS, (L >= 128 ? PA_SWEEP_MINB128 : PA_SWEEP_MINB64))
k_sweep(const DevState* __restrict__ st, uint32_t* spins0, uint32_t* spins1,
        int32_t* __restrict__ EM0, int32_t* __restrict__ EM1,
        const PhiloxKey key, const SweepArgs sa, const uint32_t* __restrict__ parent_of,
        const uint4* __restrict__ bond_mask) {
  using G_ = Geo<L>;
  static_assert(L >= 64, "k_sweep_small handles L < 64");
  grid_dependency_wait();
  if (st->status != ST_OK) return;
  const unsigned buf = (sa.mode == 1 || sa.mode == 3) ? st->cur : (st->cur ^ 1u);
  const unsigned long long count = sa.mode != 1 ? st->Rnew : st->R;
  const int theta = sa.mode != 1 ? sa.theta : 0;
  uint32_t* spins = buf ? spins1 : spins0;
  const uint32_t* spins_other = buf ? spins0 : spins1;  // buffer cur inside a step
  int32_t* __restrict__ EMo = buf ? EM1 : EM0;  // packed E/4 : M/2 words (pa_common.cuh)

  const unsigned long long slot_base64 = (unsigned long long)blockIdx.x * G_::RPB;
  if (slot_base64 >= count) return;  // block-uniform: the sweeps below contain block barriers
  const int g = (int)(threadIdx.x % G_::G);
  const unsigned long long slot0_64 = slot_base64 + (unsigned long long)(threadIdx.x / G_::G) * G_::RW;  // the warp's first replica
  const uint32_t slot0 = (uint32_t)slot0_64, slot_base = (uint32_t)slot_base64;
  bool valid[G_::RW];  // warp-uniform

  // ---- load (once per step): the lane's rows are RPL*WR contiguous words = RPL*WR/4 16-byte vectors ----
  Lattice<L> lat[G_::RW];
  constexpr int NV = G_::RPL * G_::WR / 4;
#pragma unroll
  for (int rep = 0; rep < G_::RW; ++rep) {
    const unsigned long long slot64 = slot0_64 + rep;
    valid[rep] = slot64 < count;
    const uint32_t* rep_src = spins + (valid[rep] ? slot64 : slot_base64) * G_::WREP;
    if (sa.mode == 2 && valid[rep]) rep_src = spins_other + (unsigned long long)parent_of[slot64] * G_::WREP;  // parent
    uint32_t rawall[G_::RPL * G_::WR];
    const uint4* src = reinterpret_cast<const uint4*>(rep_src) + g * NV;
#pragma unroll
    for (int v = 0; v < NV; ++v) {
      const uint4 x = src[v];
      rawall[4 * v] = x.x; rawall[4 * v + 1] = x.y; rawall[4 * v + 2] = x.z; rawall[4 * v + 3] = x.w;
    }
#pragma unroll
    for (int r = 0; r < G_::RPL; ++r) {
      uint32_t raw[G_::WR];
#pragma unroll
      for (int i = 0; i < G_::WR; ++i) raw[i] = rawall[r * G_::WR + i];
      row_to_planes<L>(raw, (g * G_::RPL + r) & 1, lat[rep].p[0][r], lat[rep].p[1][r]);
    }
  }

  // ---- theta sweeps ----------------------------------------------------------------------------
  if (theta > 0) {
    const uint32_t c3 = ctr3(TAG_SWEEP, st->step + 1u);
    const uint32_t gs = st->slot0_new;  // global index of local slot 0 (0 unless this is a multi-GPU shard)
    using Q_ = SweepQueue<SweepCap<G_::NWL>::CAP>;
    __shared__ Q_ q_mem;
    static_assert(offsetof(Q_, res) == Q_::OFF_RES && offsetof(Q_, count) == Q_::OFF_COUNT, "queue layout");
    uint32_t q = (uint32_t)__cvta_generic_to_shared(&q_mem);
    asm volatile("mov.u32 %0, %0;" : "+r"(q));  // keep it in a register: ptxas otherwise rebuilds it (S2R + LEA) at every use
    if (threadIdx.x < 2) q_mem.count[threadIdx.x] = 0u;
    queue_clear_results<G_::NWL, SWEEP_THREADS, SweepCap<G_::NWL>::CAP>(q);
    __syncthreads();
#pragma unroll 1
    for (uint32_t h = 0; h < 2u * (uint32_t)theta; ++h)  // half-sweep h = 2t + colour
      half_sweep_rt<L, SG>(lat, q, g, h & 1u, slot0 + gs, slot_base + gs, h, c3, key, sa, bond_mask);
  }

#pragma unroll
  for (int rep = 0; rep < G_::RW; ++rep) {
    if (!valid[rep]) continue;  // warp-uniform
    const unsigned long long slot64 = slot0_64 + rep;
    // ---- a8: E = 2u - 2N, M = 2*popc - N ----------------------------------------------------------
    int unsat, ups;
    count_bonds<L, SG>(lat[rep], g, bond_mask, unsat, ups);
#pragma unroll
    for (int o = G_::G / 2; o > 0; o >>= 1) {
      unsat += __shfl_xor_sync(0xffffffffu, unsat, o);
      ups += __shfl_xor_sync(0xffffffffu, ups, o);
    }
    if (g == 0) EMo[slot64] = pack_em(2 * unsat - 2 * G_::N, 2 * ups - G_::N);
    // ---- store (once per step) -------------------------------------------------------------------
    if (theta > 0) {
      uint32_t rawall[G_::RPL * G_::WR];
#pragma unroll
      for (int r = 0; r < G_::RPL; ++r) {
        uint32_t raw[G_::WR];
        planes_to_row<L>(lat[rep].p[0][r], lat[rep].p[1][r], (g * G_::RPL + r) & 1, raw);
#pragma unroll
        for (int i = 0; i < G_::WR; ++i) rawall[r * G_::WR + i] = raw[i];
      }
      uint4* dst = reinterpret_cast<uint4*>(spins + slot64 * G_::WREP) + g * NV;
#pragma unroll
      for (int v = 0; v < NV; ++v)
        dst[v] = make_uint4(rawall[4 * v], rawall[4 * v + 1], rawall[4 * v + 2], rawall[4 * v + 3]);
    }
  }
}

// =====================================================================================================
// L < 64: one plane word = RG = 64/L consecutive rows of HB = L/2 bits; a replica is G = N/64 lanes with one
// word per colour each (L = 32: 16 lanes, L = 16: 4 lanes, L = 8: one thread holds the whole replica).
// =====================================================================================================
template <int L>
struct SGeo {
  static constexpr int N = L * L;
  static constexpr int G = N / 64;      // lanes per replica
  static constexpr int HB = L / 2;      // bits per row field
  static constexpr int RG = 32 / HB;    // rows per word (even)
  static constexpr int WREP = N / 32;
  static constexpr uint32_t FIELD = (1u << HB) - 1u;
  static constexpr uint32_t ER = L == 32 ? 0x0000ffffu : (L == 16 ? 0x00ff00ffu : 0x0f0f0f0fu);   // fields of even rows
  static constexpr uint32_t LSBS = L == 32 ? 0x00010001u : (L == 16 ? 0x01010101u : 0x11111111u);  // bit 0 of every field
  static constexpr uint32_t MSBS = LSBS << (HB - 1);
};

template <int L, int NR>
struct SmallSlotOf {
  static __device__ __forceinline__ uint32_t rel(unsigned t, unsigned w) { return (t / (unsigned)SGeo<L>::G) * (unsigned)NR + w; }
};

// neighbour words of the lane's word of plane C: S = the lane's word of plane 1-C
template <int L, int C>
__device__ __forceinline__ void small_neighbours(uint32_t S, int g, uint32_t& U, uint32_t& D, uint32_t& B) {
  using G_ = SGeo<L>;
  uint32_t Sp = S, Sn = S;
  if constexpr (G_::G > 1) {
    Sp = __shfl_sync(0xffffffffu, S, (g + G_::G - 1) % G_::G, G_::G);
    Sn = __shfl_sync(0xffffffffu, S, (g + 1) % G_::G, G_::G);
  }
  U = __funnelshift_l(Sp, S, G_::HB);  // row y-1 at the position of row y: (S << HB) | (Sp >> (32 - HB))
  D = __funnelshift_r(S, Sn, G_::HB);  // row y+1:                          (S >> HB) | (Sn << (32 - HB))
  const uint32_t rotl = ((S << 1) & ~G_::LSBS) | ((S >> (G_::HB - 1)) & G_::LSBS);  // bit k <- bit k-1 inside every field
  const uint32_t rotr = ((S >> 1) & ~G_::MSBS) | ((S << (G_::HB - 1)) & G_::MSBS);  // bit k <- bit k+1
  // row y uses k-1 when (y + C) is even; the word's first row is even
  B = C == 0 ? ((rotl & G_::ER) | (rotr & ~G_::ER)) : ((rotr & G_::ER) | (rotl & ~G_::ER));
}

// NR = replicas per lane group: 2 for small populations (more blocks: config 1 is latency-bound), 8 for large ones (8
// plane words per lane and half-sweep, as in k_sweep: specialised comparator, region-form queue, per-word overheads
// amortised)
template <int L, bool SG, int NR>
__global__ void __launch_bounds__(SWEEP_SMALL_THREADS, NR >= 8 ? 4 : 5)
k_sweep_small(const DevState* __restrict__ st, uint32_t* spins0, uint32_t* spins1,
              int32_t* __restrict__ EM0, int32_t* __restrict__ EM1,
              const PhiloxKey key, const SweepArgs sa, const uint32_t* __restrict__ parent_of,
              const uint4* __restrict__ bond_mask) {
  using G_ = SGeo<L>;
  static_assert(L == 8 || L == 16 || L == 32, "");
  grid_dependency_wait();
  if (st->status != ST_OK) return;
  const unsigned buf = (sa.mode == 1 || sa.mode == 3) ? st->cur : (st->cur ^ 1u);
  const unsigned long long count = sa.mode != 1 ? st->Rnew : st->R;
  const int theta = sa.mode != 1 ? sa.theta : 0;
  uint32_t* spins = buf ? spins1 : spins0;
  int32_t* __restrict__ EMo = buf ? EM1 : EM0;  // packed E/4 : M/2 words (pa_common.cuh)
  const uint32_t gs = sa.mode != 1 ? st->slot0_new : 0u;  // global index of local slot 0 (multi-GPU shard)

  // A group of G lanes holds NR consecutive replicas (one plane word per colour and replica per lane).
  const unsigned long long tid = (unsigned long long)blockIdx.x * SWEEP_SMALL_THREADS + threadIdx.x;
  const unsigned long long pair = tid / G_::G;
  const int g = (int)(tid % G_::G);
  const unsigned long long slot_base64 = ((unsigned long long)blockIdx.x * SWEEP_SMALL_THREADS / G_::G) * NR;
  if (slot_base64 >= count) return;  // block-uniform: the sweeps below contain block barriers
  uint4 mk[2] = {make_uint4(0u, 0u, 0u, 0u), make_uint4(0u, 0u, 0u, 0u)};  // negative bonds of the lane's word, per colour
  if constexpr (SG) {
    mk[0] = __ldg(bond_mask + g);
    mk[1] = __ldg(bond_mask + G_::G + g);
  }
  const uint32_t slot_base = (uint32_t)slot_base64;
  const unsigned long long slot0_64 = pair * NR;  // the group's first replica; slot r of the group is slot0_64 + r
  uint32_t slots[NR];
  uint32_t p[NR][2];
#pragma unroll
  for (int r = 0; r < NR; ++r) {
    const unsigned long long slot64 = slot0_64 + r;
    const bool valid = slot64 < count;
    slots[r] = (uint32_t)slot64 + gs;
    const uint32_t* rep_src = spins + (valid ? slot64 : 0ull) * G_::WREP;
    if (sa.mode == 2 && valid) rep_src = (buf ? spins0 : spins1) + (unsigned long long)parent_of[slot64] * G_::WREP;
    // ---- load: 64 raw bits = RG rows -------------------------------------------------------------
    const uint2 q = valid ? reinterpret_cast<const uint2*>(rep_src)[g] : make_uint2(0u, 0u);
    const uint32_t ev = even_bits(q.x) | (even_bits(q.y) << 16);
    const uint32_t od = even_bits(q.x >> 1) | (even_bits(q.y >> 1) << 16);
    p[r][0] = (ev & G_::ER) | (od & ~G_::ER);  // even row: colour 0 sits at even x; odd row: at odd x
    p[r][1] = (od & G_::ER) | (ev & ~G_::ER);
  }

  // ---- theta sweeps ----------------------------------------------------------------------------
  if (theta > 0) {
    using Q_ = SweepQueue<SweepCap<NR, SWEEP_SMALL_THREADS>::CAP>;
    __shared__ Q_ q_mem;
    static_assert(offsetof(Q_, res) == Q_::OFF_RES && offsetof(Q_, count) == Q_::OFF_COUNT, "queue layout");
    uint32_t q = (uint32_t)__cvta_generic_to_shared(&q_mem);
    asm volatile("mov.u32 %0, %0;" : "+r"(q));  // keep it in a register: ptxas otherwise rebuilds it (S2R + LEA) at every use
    if (threadIdx.x < 2) q_mem.count[threadIdx.x] = 0u;
    queue_clear_results<NR, SWEEP_SMALL_THREADS, SweepCap<NR, SWEEP_SMALL_THREADS>::CAP>(q);
    __syncthreads();
    const uint32_t c3 = ctr3(TAG_SWEEP, st->step + 1u);
    uint32_t call0[NR];
#pragma unroll
    for (int r = 0; r < NR; ++r) call0[r] = 8u * (uint32_t)g;  // group = g
    for (int t = 0; t < theta; ++t) {
      {
        uint32_t ge1[NR], ge2[NR], flip[NR];
#pragma unroll
        for (int r = 0; r < NR; ++r) {
          uint32_t U, D, B;
          small_neighbours<L, 0>(p[r][1], g, U, D, B);
          neighbour_classes_j<SG>(p[r][0], U, D, p[r][1], B, mk[0], ge1[r], ge2[r]);
        }
        queued_accept<NR, SWEEP_SMALL_THREADS, SweepCap<NR, SWEEP_SMALL_THREADS>::CAP, SmallSlotOf<L, NR>>(q, 0u, ge1, ge2, slots, slot_base + gs, call0, 2u * (uint32_t)t, c3, key,
                                                           sa, flip);
#pragma unroll
        for (int r = 0; r < NR; ++r) p[r][0] ^= flip[r];
      }
      {
        uint32_t ge1[NR], ge2[NR], flip[NR];
#pragma unroll
        for (int r = 0; r < NR; ++r) {
          uint32_t U, D, B;
          small_neighbours<L, 1>(p[r][0], g, U, D, B);
          neighbour_classes_j<SG>(p[r][1], U, D, p[r][0], B, mk[1], ge1[r], ge2[r]);
        }
        queued_accept<NR, SWEEP_SMALL_THREADS, SweepCap<NR, SWEEP_SMALL_THREADS>::CAP, SmallSlotOf<L, NR>>(q, 1u, ge1, ge2, slots, slot_base + gs, call0, 2u * (uint32_t)t + 1u, c3,
                                                           key, sa, flip);
#pragma unroll
        for (int r = 0; r < NR; ++r) p[r][1] ^= flip[r];
      }
    }
  }

#pragma unroll
  for (int r = 0; r < NR; ++r) {
    // ---- a8: every bond has exactly one colour-0 end ----------------------------------------------
    uint32_t U, D, B;
    small_neighbours<L, 0>(p[r][1], g, U, D, B);
    int unsat = __popc(p[r][0] ^ U ^ mk[0].x) + __popc(p[r][0] ^ D ^ mk[0].y) + __popc(p[r][0] ^ p[r][1] ^ mk[0].z) +
                __popc(p[r][0] ^ B ^ mk[0].w);
    int ups = __popc(p[r][0]) + __popc(p[r][1]);
#pragma unroll
    for (int o = G_::G / 2; o > 0; o >>= 1) {
      unsat += __shfl_xor_sync(0xffffffffu, unsat, o);
      ups += __shfl_xor_sync(0xffffffffu, ups, o);
    }
    const unsigned long long slot64 = slot0_64 + r;
    const bool valid = slot64 < count;
    if (valid && g == 0) EMo[slot64] = pack_em(2 * unsat - 2 * G_::N, 2 * ups - G_::N);
    // ---- store -----------------------------------------------------------------------------------
    if (theta > 0 && valid) {
      const uint32_t ev = (p[r][0] & G_::ER) | (p[r][1] & ~G_::ER);
      const uint32_t od = (p[r][1] & G_::ER) | (p[r][0] & ~G_::ER);
      uint2 q;
      q.x = spread_bits(ev) | (spread_bits(od) << 1);
      q.y = spread_bits(ev >> 16) | (spread_bits(od >> 16) << 1);
      reinterpret_cast<uint2*>(spins + slot64 * G_::WREP)[g] = q;
    }
  }
}

}  // namespace pa
