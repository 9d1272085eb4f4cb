// pa_sweep.cuh -- a7/a8: theta checkerboard Metropolis sweeps of every replica + E, M from the final lattice.
// PAPER.md:56 (MCMC equilibration at the new temperature), :126-128 (theta), :62 (observables);
// rule and random keying: DESIGN.md "C3", "C4".
//
// Layout in registers (multispin coding WITHIN a replica): G = min(L,32) lanes share one replica, lane g holds
// rows g*RPL .. g*RPL+RPL-1.  Every row is split into its two colour planes so that one 32-bit word holds 32
// sites that are updated simultaneously:
//   plane c of row y, bit k  <->  site x = 2k + ((y + c) & 1)          (colour (x+y)&1 == c)
// The four neighbours of a colour-c site (k,y) are colour 1-c sites: rows y-1, y+1 at bit k, row y at bit k,
// and row y at bit k-1 (if (y+c) even) or k+1 (if odd), all modulo L/2.  Up/down rows of neighbouring lanes
// come by warp shuffle.  The lattice is read from HBM once and written once per step; nothing else touches
// memory during the theta sweeps.
#pragma once
#include "pa_common.cuh"

namespace pa {

template <int L>
struct Geo {
  static constexpr int N = L * L;
  static constexpr int G = L < 32 ? L : 32;       // lanes per replica
  static constexpr int RPL = L / G;               // rows per lane
  static constexpr int HB = L / 2;                // bits per row per colour plane
  static constexpr int WPP = (HB + 31) / 32;      // words per row plane
  static constexpr int WR = (L + 31) / 32;        // raw words per row
  static constexpr int WREP = N / 32;             // words per replica
  static constexpr int NB = HB < 32 ? HB : 32;    // used bits per plane word
  static constexpr uint32_t HMASK = HB >= 32 ? 0xffffffffu : ((1u << (HB & 31)) - 1u);
  static constexpr int CALLS_PER_WORD = NB / 4;   // Philox blocks per plane word
  static constexpr int CALLS_PER_ROW = HB / 4;
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

// acc |= BIT if w < T (unsigned).  Written as compare + predicated OR so that both instructions stay on the
// ALU pipe: the FMA pipe is saturated by Philox's 32x32->64 multiplies (ptxas turns carry-based forms into IMAD.X).
template <uint32_t BIT>
__device__ __forceinline__ void or_if_lt(uint32_t& acc, uint32_t w, uint32_t T) {
  asm("{\n\t.reg .pred p;\n\tsetp.lt.u32 p, %1, %2;\n\t@p or.b32 %0, %0, %3;\n\t}" : "+r"(acc) : "r"(w), "r"(T), "n"(BIT));
}

// the two random masks of one Philox block (4 consecutive active sites) at bit offset SH
template <int SH>
__device__ __forceinline__ void push_block(uint32_t& r4, uint32_t& r8, const uint4& w, uint32_t T4, uint32_t T8) {
  or_if_lt<(1u << SH)>(r4, w.x, T4); or_if_lt<(2u << SH)>(r4, w.y, T4);
  or_if_lt<(4u << SH)>(r4, w.z, T4); or_if_lt<(8u << SH)>(r4, w.w, T4);
  or_if_lt<(1u << SH)>(r8, w.x, T8); or_if_lt<(2u << SH)>(r8, w.y, T8);
  or_if_lt<(4u << SH)>(r8, w.z, T8); or_if_lt<(8u << SH)>(r8, w.w, T8);
}

template <int L>
struct Lattice {
  using G_ = Geo<L>;
  uint32_t p[2][G_::RPL][G_::WPP];  // colour planes
};

// rotate plane row so that result bit k = source bit k-1 (dir = 0) or k+1 (dir = 1), modulo HB
template <int L>
__device__ __forceinline__ void rot_row(const uint32_t (&s)[Geo<L>::WPP], int dir, uint32_t (&out)[Geo<L>::WPP]) {
  using G_ = Geo<L>;
  if constexpr (G_::HB >= 32) {
#pragma unroll
    for (int i = 0; i < G_::WPP; ++i) {
      const uint32_t prev = s[(i + G_::WPP - 1) % G_::WPP], next = s[(i + 1) % G_::WPP];
      const uint32_t left = __funnelshift_l(prev, s[i], 1);   // (s[i] << 1) | (prev >> 31)
      const uint32_t right = __funnelshift_r(s[i], next, 1);  // (s[i] >> 1) | (next << 31)
      out[i] = dir ? right : left;
    }
  } else {
    const uint32_t a = s[0];
    const uint32_t left = ((a << 1) | (a >> (G_::HB - 1))) & G_::HMASK;
    const uint32_t right = ((a >> 1) | (a << (G_::HB - 1))) & G_::HMASK;
    out[0] = dir ? right : left;
  }
}

// One half-sweep of colour C on the lane's rows.  T = plane C (updated), S = plane 1-C (read only).
template <int L, int C>
__device__ __forceinline__ void half_sweep(Lattice<L>& lat, int g, uint32_t slot, uint32_t t, uint32_t c3,
                                           const PhiloxKey& key, uint32_t T4, uint32_t T8) {
  using G_ = Geo<L>;
  constexpr unsigned FULL = 0xffffffffu;
  uint32_t(&T)[G_::RPL][G_::WPP] = lat.p[C];
  uint32_t(&S)[G_::RPL][G_::WPP] = lat.p[1 - C];
  // rows above the lane's first row and below its last row
  uint32_t up[G_::WPP], dn[G_::WPP];
  const int gu = (g + G_::G - 1) % G_::G, gd = (g + 1) % G_::G;
#pragma unroll
  for (int i = 0; i < G_::WPP; ++i) {
    up[i] = __shfl_sync(FULL, S[G_::RPL - 1][i], gu, G_::G);
    dn[i] = __shfl_sync(FULL, S[0][i], gd, G_::G);
  }
  const uint32_t c2 = 2u * t + (uint32_t)C;
#pragma unroll
  for (int r = 0; r < G_::RPL; ++r) {
    const int y = g * G_::RPL + r;
    const int dir = (y + C) & 1;
    uint32_t B[G_::WPP];
    rot_row<L>(S[r], dir, B);
#pragma unroll
    for (int i = 0; i < G_::WPP; ++i) {
      const uint32_t U = (r > 0) ? S[r > 0 ? r - 1 : 0][i] : up[i];
      const uint32_t D = (r < G_::RPL - 1) ? S[r < G_::RPL - 1 ? r + 1 : 0][i] : dn[i];
      const uint32_t tt = T[r][i];
      const uint32_t d0 = tt ^ U, d1 = tt ^ D, d2 = tt ^ S[r][i], d3 = tt ^ B[i];  // 1 = anti-aligned
      const uint32_t maj = (d0 & d1) | (d0 & d2) | (d1 & d2);
      const uint32_t any3 = d0 | d1 | d2;
      const uint32_t ge2 = maj | (any3 & d3);  // a >= 2: dE <= 0, always flip
      const uint32_t ge1 = any3 | d3;
      // random masks: bit k set iff the site's keyed word < T4 (resp. T8)
      uint32_t r4 = 0u, r8 = 0u;
      const uint32_t call0 = (uint32_t)y * G_::CALLS_PER_ROW + (uint32_t)i * 8u;
      if constexpr (G_::RPL * G_::WPP <= 2) {
        // small lattices per lane: fully unrolled, bit positions are immediates
#pragma unroll
        for (int cc = 0; cc < G_::CALLS_PER_WORD; ++cc) {
          const uint4 w = philox4x32_10(slot, call0 + cc, c2, c3, key);
          switch (cc) {
            case 0: push_block<0>(r4, r8, w, T4, T8); break;
            case 1: push_block<4>(r4, r8, w, T4, T8); break;
            case 2: push_block<8>(r4, r8, w, T4, T8); break;
            case 3: push_block<12>(r4, r8, w, T4, T8); break;
            case 4: push_block<16>(r4, r8, w, T4, T8); break;
            case 5: push_block<20>(r4, r8, w, T4, T8); break;
            case 6: push_block<24>(r4, r8, w, T4, T8); break;
            default: push_block<28>(r4, r8, w, T4, T8); break;
          }
        }
      } else {
        // L = 128: 8 plane words per lane; keep the block loop rolled (two chains in flight) to bound code size
#pragma unroll 2
        for (int cc = 0; cc < G_::CALLS_PER_WORD; ++cc) {
          const uint4 w = philox4x32_10(slot, call0 + cc, c2, c3, key);
          uint32_t n4 = 0u, n8 = 0u;
          push_block<0>(n4, n8, w, T4, T8);
          r4 |= n4 << (4 * cc);
          r8 |= n8 << (4 * cc);
        }
      }
      // flip iff a>=2, or a==1 and u<T4, or a==0 and u<T8
      const uint32_t flip = ge2 | (ge1 & r4) | (~ge1 & r8);
      T[r][i] = tt ^ flip;
    }
  }
}

// number of anti-aligned bonds u (each bond has exactly one colour-0 end) and number of up spins
template <int L>
__device__ __forceinline__ void count_bonds(const Lattice<L>& lat, int g, int& unsat, int& ups) {
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
      u += __popc(tt ^ U) + __popc(tt ^ D) + __popc(tt ^ S[r][i]) + __popc(tt ^ B[i]);
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
  uint32_t ev[G_::WPP], od[G_::WPP];
  if constexpr (L >= 64) {
#pragma unroll
    for (int i = 0; i < G_::WPP; ++i) {
      ev[i] = even_bits(raw[2 * i]) | (even_bits(raw[2 * i + 1]) << 16);
      od[i] = even_bits(raw[2 * i] >> 1) | (even_bits(raw[2 * i + 1] >> 1) << 16);
    }
  } else {
    ev[0] = even_bits(raw[0]);
    od[0] = even_bits(raw[0] >> 1);
  }
#pragma unroll
  for (int i = 0; i < G_::WPP; ++i) {  // even row: colour 0 sits at even x; odd row: at odd x
    p0[i] = y_odd ? od[i] : ev[i];
    p1[i] = y_odd ? ev[i] : od[i];
  }
}
template <int L>
__device__ __forceinline__ void planes_to_row(const uint32_t (&p0)[Geo<L>::WPP], const uint32_t (&p1)[Geo<L>::WPP],
                                              int y_odd, uint32_t (&raw)[Geo<L>::WR]) {
  using G_ = Geo<L>;
#pragma unroll
  for (int i = 0; i < G_::WPP; ++i) {
    const uint32_t ev = y_odd ? p1[i] : p0[i], od = y_odd ? p0[i] : p1[i];
    if constexpr (L >= 64) {
      raw[2 * i] = spread_bits(ev) | (spread_bits(od) << 1);
      raw[2 * i + 1] = spread_bits(ev >> 16) | (spread_bits(od >> 16) << 1);
    } else {
      raw[0] = spread_bits(ev) | (spread_bits(od) << 1);
    }
  }
}

constexpr int SWEEP_THREADS = 256;

// mode 0: inside a step -> buffer cur^1, Rnew replicas, theta sweeps keyed with step ordinal st->step+1
// mode 1: init / set_spins -> buffer cur, R replicas, no sweeps (energies only)
template <int L>
__global__ void __launch_bounds__(SWEEP_THREADS, (L >= 128 ? 2 : 3))
k_sweep(const DevState* __restrict__ st, const StepParams* __restrict__ sp, uint32_t* __restrict__ spins0,
        uint32_t* __restrict__ spins1, int32_t* __restrict__ E0, int32_t* __restrict__ E1, int32_t* __restrict__ M0,
        int32_t* __restrict__ M1, const PhiloxKey key, const int mode) {
  using G_ = Geo<L>;
  if (st->status != ST_OK) return;
  const unsigned buf = mode == 0 ? (st->cur ^ 1u) : st->cur;
  const unsigned long long count = mode == 0 ? st->Rnew : st->R;
  const int theta = mode == 0 ? sp->theta : 0;
  uint32_t* __restrict__ spins = buf ? spins1 : spins0;
  int32_t* __restrict__ Eo = buf ? E1 : E0;
  int32_t* __restrict__ Mo = buf ? M1 : M0;

  const unsigned long long tid = (unsigned long long)blockIdx.x * SWEEP_THREADS + threadIdx.x;
  const unsigned long long slot64 = tid / G_::G;
  const int g = (int)(tid % G_::G);
  {  // warp-uniform exit for warps entirely past the population
    const unsigned long long first_slot_of_warp = (tid & ~31ull) / G_::G;
    if (first_slot_of_warp >= count) return;
  }
  const bool valid = slot64 < count;
  const uint32_t slot = (uint32_t)slot64;
  uint32_t* rep = spins + (valid ? slot64 : 0ull) * G_::WREP;

  // ---- load (once per step) -------------------------------------------------------------------
  Lattice<L> lat;
  if constexpr (L >= 64) {
    // lane's rows are RPL*WR contiguous words = RPL*WR/4 16-byte vectors
    constexpr int NV = G_::RPL * G_::WR / 4;
    uint32_t rawall[G_::RPL * G_::WR];
    const uint4* src = reinterpret_cast<const uint4*>(rep) + g * NV;
#pragma unroll
    for (int v = 0; v < NV; ++v) {
      const uint4 q = valid ? src[v] : make_uint4(0, 0, 0, 0);
      rawall[4 * v] = q.x; rawall[4 * v + 1] = q.y; rawall[4 * v + 2] = q.z; rawall[4 * v + 3] = q.w;
    }
#pragma unroll
    for (int r = 0; r < G_::RPL; ++r) {
      uint32_t raw[G_::WR];
#pragma unroll
      for (int i = 0; i < G_::WR; ++i) raw[i] = rawall[r * G_::WR + i];
      row_to_planes<L>(raw, (g * G_::RPL + r) & 1, lat.p[0][r], lat.p[1][r]);
    }
  } else {
    // one row per lane; 32/L rows share a word
    constexpr int RW = 32 / L;
    const uint32_t word = valid ? rep[g / RW] : 0u;
    uint32_t raw[1];
    raw[0] = (L == 32) ? word : ((word >> ((g % RW) * L)) & ((1u << (L & 31)) - 1u));
    row_to_planes<L>(raw, g & 1, lat.p[0][0], lat.p[1][0]);
  }

  // ---- theta sweeps ----------------------------------------------------------------------------
  if (theta > 0) {
    const uint32_t c3 = ctr3(TAG_SWEEP, st->step + 1u);
    const uint32_t T4 = sp->T4, T8 = sp->T8;
    for (int t = 0; t < theta; ++t) {
      half_sweep<L, 0>(lat, g, slot, (uint32_t)t, c3, key, T4, T8);
      half_sweep<L, 1>(lat, g, slot, (uint32_t)t, c3, key, T4, T8);
    }
  }

  // ---- a8: E = 2u - 2N, M = 2*popc - N ----------------------------------------------------------
  int unsat, ups;
  count_bonds<L>(lat, g, unsat, ups);
#pragma unroll
  for (int o = G_::G / 2; o > 0; o >>= 1) {
    unsat += __shfl_xor_sync(0xffffffffu, unsat, o);
    ups += __shfl_xor_sync(0xffffffffu, ups, o);
  }
  if (valid && g == 0) {
    Eo[slot64] = 2 * unsat - 2 * G_::N;
    Mo[slot64] = 2 * ups - G_::N;
  }

  // ---- store (once per step) -------------------------------------------------------------------
  if (theta > 0) {
    if constexpr (L >= 64) {
      constexpr int NV = G_::RPL * G_::WR / 4;
      uint32_t rawall[G_::RPL * G_::WR];
#pragma unroll
      for (int r = 0; r < G_::RPL; ++r) {
        uint32_t raw[G_::WR];
        planes_to_row<L>(lat.p[0][r], lat.p[1][r], (g * G_::RPL + r) & 1, raw);
#pragma unroll
        for (int i = 0; i < G_::WR; ++i) rawall[r * G_::WR + i] = raw[i];
      }
      uint4* dst = reinterpret_cast<uint4*>(rep) + g * NV;
      if (valid) {
#pragma unroll
        for (int v = 0; v < NV; ++v)
          dst[v] = make_uint4(rawall[4 * v], rawall[4 * v + 1], rawall[4 * v + 2], rawall[4 * v + 3]);
      }
    } else {
      constexpr int RW = 32 / L;
      uint32_t raw[1];
      planes_to_row<L>(lat.p[0][0], lat.p[1][0], g & 1, raw);
      uint32_t word = (L == 32) ? raw[0] : (raw[0] << ((g % RW) * L));
#pragma unroll
      for (int o = 1; o < RW; o <<= 1) word |= __shfl_xor_sync(0xffffffffu, word, o);
      if (valid && (g % RW) == 0) rep[g / RW] = word;
    }
  }
}

}  // namespace pa
