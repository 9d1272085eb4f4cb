// pa_observe.cuh -- a0 initial population and a8 population sums + commit of the step.
#pragma once
#include "pa_common.cuh"

namespace pa {

// a0: uint32 word v of replica j <- w[v&3] of Philox counter (v>>2, j, 0, tag0|0)   (C3 init)
// One thread per Philox block = up to 4 consecutive words.
__global__ void k_init(const DevState* __restrict__ st, uint32_t* __restrict__ spins0, uint32_t* __restrict__ spins1,
                       int wrep, const PhiloxKey key) {
  const unsigned long long R = st->R;
  uint32_t* __restrict__ spins = st->cur ? spins1 : spins0;
  const int blocks_per_rep = (wrep + 3) / 4;
  const unsigned long long idx = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
  const unsigned long long j = idx / blocks_per_rep;
  const unsigned b = (unsigned)(idx % blocks_per_rep);
  if (j >= R) return;
  const uint4 w = philox4x32_10(b, (uint32_t)j + st->slot0, 0u, ctr3(TAG_INIT, 0u), key);  // keyed by the GLOBAL replica index
  uint32_t* dst = spins + j * wrep + 4 * b;
  if (wrep - 4 * (int)b >= 4) {
    *reinterpret_cast<uint4*>(dst) = w;
  } else {
    const uint32_t ww[4] = {w.x, w.y, w.z, w.w};
    for (int i = 0; i < wrep - 4 * (int)b; ++i) dst[i] = ww[i];
  }
}

// getters: packed E/4 : M/2 words -> separate int32 arrays
__global__ void k_unpack_em(const int32_t* __restrict__ EM, int32_t* __restrict__ E, int32_t* __restrict__ M,
                            unsigned long long n, int e_off) {
  const unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const int32_t w = EM[i];
  if (E) E[i] = em_energy(w, e_off);
  if (M) M[i] = em_mag(w);
}

// 128-bit unsigned add helper on {lo, hi}
struct U128 {
  unsigned long long lo, hi;
};
__device__ __forceinline__ void u128_add(U128& a, unsigned long long lo, unsigned long long hi) {
  const unsigned long long s = a.lo + lo;
  a.hi += hi + (s < a.lo ? 1ull : 0ull);
  a.lo = s;
}
__device__ __forceinline__ U128 warp_sum_u128(U128 v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    const unsigned long long lo = __shfl_xor_sync(0xffffffffu, v.lo, o);
    const unsigned long long hi = __shfl_xor_sync(0xffffffffu, v.hi, o);
    u128_add(v, lo, hi);
  }
  return v;
}

// ---------------------------------------------------------------------------------------------------
// balance_tile: a5.  One block (the last block of k_observe: every offset of the step is in memory).  New partition
// table, born/excess/shortage per partition, moved count.  PAPER.md:84-118; A6, A6b (readings G21-G23).
//   policy 0  balanced: cnt_p = floor(R'/P) + (p < R' mod P)           (any P)
//   policy 1  main:     blocks of B replicas move from the largest excess to the largest shortage until every partition
//                       is within maxexc blocks of its balanced count
//   policy 2  naive:    every partition pools floor(born_p / 2), the pool is dealt back evenly
//   policy 3  none:     cnt_p = born_p
// Policies 1-3 keep the partition counts in shared memory (P <= BAL_PMAX).
// ---------------------------------------------------------------------------------------------------
constexpr int BAL_PMAX = 1024;

struct BalanceArgs {
  int P, policy;
  unsigned B, maxexc;
};

__device__ void balance_tile(DevState* st, const uint32_t* off, uint32_t* part0, uint32_t* part1, uint32_t* stats,
                             const BalanceArgs ba) {
  if (*((volatile unsigned*)&st->status) != ST_OK) return;
  const int P = ba.P;
  const uint32_t* old_start = st->cur ? part1 : part0;
  uint32_t* new_start = st->cur ? part0 : part1;
  const unsigned long long Rnew = *((volatile unsigned long long*)&st->Rnew);
  const unsigned long long base = Rnew / P, rem = Rnew % P;
  __shared__ unsigned long long s_same;
  __shared__ long long s_c[BAL_PMAX];        // counts of policies 1-3
  __shared__ uint32_t s_start[BAL_PMAX + 1];
  if (threadIdx.x == 0) s_same = 0ull;
  if (ba.policy != 0) {
    for (int p = threadIdx.x; p < P; p += blockDim.x)
      s_c[p] = (long long)__ldcg(off + old_start[p + 1]) - (long long)__ldcg(off + old_start[p]);  // born_p
    __syncthreads();
    if (ba.policy == 2 && threadIdx.x == 0) {
      long long pool = 0;
      for (int p = 0; p < P; ++p) pool += s_c[p] / 2;
      const long long share = pool / P, extra = pool % P;
      for (int p = 0; p < P; ++p) s_c[p] = s_c[p] - s_c[p] / 2 + share + (p < extra ? 1 : 0);
    }
    if (ba.policy == 1 && threadIdx.x < 32) {  // warp 0: one block move per iteration
      const long long W = (long long)ba.maxexc * (long long)ba.B;
      const int lane = threadIdx.x;
      for (;;) {
        long long e_hi = 0, e_lo = 0;
        int hi = -1, lo = -1;
        for (int p = lane; p < P; p += 32) {  // ascending p: strict comparisons keep the lowest index on ties
          const long long e = s_c[p] - (long long)(base + ((unsigned long long)p < rem ? 1ull : 0ull));
          if (hi < 0 || e > e_hi) { e_hi = e; hi = p; }
          if (lo < 0 || e < e_lo) { e_lo = e; lo = p; }
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
          const long long oe_hi = __shfl_xor_sync(0xffffffffu, e_hi, o), oe_lo = __shfl_xor_sync(0xffffffffu, e_lo, o);
          const int ohi = __shfl_xor_sync(0xffffffffu, hi, o), olo = __shfl_xor_sync(0xffffffffu, lo, o);
          if (ohi >= 0 && (hi < 0 || oe_hi > e_hi || (oe_hi == e_hi && ohi < hi))) { e_hi = oe_hi; hi = ohi; }
          if (olo >= 0 && (lo < 0 || oe_lo < e_lo || (oe_lo == e_lo && olo < lo))) { e_lo = oe_lo; lo = olo; }
        }
        if (e_hi <= W && -e_lo <= W) break;  // every partition inside the window
        if (lane == 0) {
          s_c[hi] -= (long long)ba.B;
          s_c[lo] += (long long)ba.B;
        }
        __syncwarp();
      }
    }
    __syncthreads();
    if (threadIdx.x == 0) {
      unsigned long long run = 0;
      for (int p = 0; p < P; ++p) {
        s_start[p] = (uint32_t)run;
        run += (unsigned long long)s_c[p];
      }
      s_start[P] = (uint32_t)run;
    }
  }
  __syncthreads();
  unsigned long long same = 0;
  for (int p = threadIdx.x; p <= P; p += blockDim.x) {
    const unsigned long long s =
        ba.policy != 0 ? s_start[p] : (unsigned long long)p * base + ((unsigned long long)p < rem ? p : rem);
    new_start[p] = (uint32_t)s;
    if (p < P) {
      const unsigned long long e = ba.policy != 0 ? s_start[p + 1]
                                                  : (unsigned long long)(p + 1) * base + ((unsigned long long)(p + 1) < rem ? p + 1 : rem);
      const uint32_t cnt = (uint32_t)(e - s);
      const uint32_t b0 = __ldcg(off + old_start[p]), b1 = __ldcg(off + old_start[p + 1]);
      const uint32_t born = b1 - b0;
      stats[4 * p + 0] = cnt;
      stats[4 * p + 1] = born;
      stats[4 * p + 2] = born > cnt ? born - cnt : 0u;
      stats[4 * p + 3] = cnt > born ? cnt - born : 0u;
      // children of partition p's parents occupy [b0, b1); those inside [s, e) stay in partition p
      const unsigned long long lo = b0 > s ? b0 : s, hi = b1 < e ? b1 : e;
      if (hi > lo) same += hi - lo;
    }
  }
  atomicAdd(&s_same, same);
  __syncthreads();
  if (threadIdx.x == 0) st->moved = Rnew - s_same;
}

constexpr int OBS_THREADS = 256;
constexpr int OBS_Q = 5;  // sum E (two's complement), sum E^2, sum |M|, sum M^2, sum M^4

// mode 0: end of a step -> sums over buffer cur^1 (Rnew replicas), then COMMIT the step.
// mode 1: after init / set_spins -> sums over buffer cur (R replicas), no commit.
// mode 2: end of a step of a multi-GPU shard -> the exchange has put the new local population (Rnew replicas) into
//         buffer cur itself; sums over it, then COMMIT without flipping the buffers.
__global__ void __launch_bounds__(OBS_THREADS)
k_observe(DevState* st, const StepParams* __restrict__ sp, const int32_t* __restrict__ EM0,
          const int32_t* __restrict__ EM1,
          unsigned long long* __restrict__ partial /* [grid][12] */, const int mode, const int N,
          const uint32_t* __restrict__ off, uint32_t* part0, uint32_t* part1, uint32_t* part_stats, const BalanceArgs ba) {
  grid_dependency_wait();
  if (st->status != ST_OK) return;
  const unsigned buf = mode == 0 ? (st->cur ^ 1u) : st->cur;
  const unsigned long long count = mode != 1 ? st->Rnew : st->R;
  const int32_t* __restrict__ EM = buf ? EM1 : EM0;  // packed E/4 : M/2 words (pa_common.cuh)
  // per-thread partial sums: a thread sees at most cap / (grid * 256) < 2^17 replicas, |E| <= 2^15, |M| <= 2^14, so
  // sum E, sum E^2 (< 2^47), sum |M|, sum M^2 fit 64 bits; only M^4 (< 2^56 each) needs the 128-bit accumulator.
  long long sE = 0;
  unsigned long long sE2 = 0, sA = 0, sM2 = 0;
  U128 sM4 = {0ull, 0ull};
  int emin = 0x7fffffff, emax = -0x7fffffff;  // occupied energy range: the level window of the next step's tables
  const int e_off = st->e_off;
  auto add = [&](int w) {
    const int ei = em_energy(w, e_off), mi = em_mag(w);
    emin = min(emin, ei);
    emax = max(emax, ei);
    const long long e = ei;
    const unsigned long long am = (unsigned long long)(mi < 0 ? -mi : mi), m2 = am * am;
    sE += e;
    sE2 += (unsigned long long)(e * e);
    sA += am;
    sM2 += m2;
    u128_add(sM4, m2 * m2, 0ull);
  };
  const unsigned long long nvec = count / 4, tid = (unsigned long long)blockIdx.x * OBS_THREADS + threadIdx.x;
  const unsigned long long stride = (unsigned long long)gridDim.x * OBS_THREADS;
  const int4* __restrict__ EM4 = reinterpret_cast<const int4*>(EM);  // buffers are 256-byte aligned
  unsigned long long v = tid;
  for (; v + 3 * stride < nvec; v += 4 * stride) {  // 64 bytes in flight per thread
    const int4 a = __ldg(EM4 + v), b = __ldg(EM4 + v + stride), c = __ldg(EM4 + v + 2 * stride), d = __ldg(EM4 + v + 3 * stride);
    add(a.x); add(a.y); add(a.z); add(a.w);
    add(b.x); add(b.y); add(b.z); add(b.w);
    add(c.x); add(c.y); add(c.z); add(c.w);
    add(d.x); add(d.y); add(d.z); add(d.w);
  }
  for (; v < nvec; v += stride) {
    const int4 a = __ldg(EM4 + v);
    add(a.x); add(a.y); add(a.z); add(a.w);
  }
  for (unsigned long long j = 4 * nvec + tid; j < count; j += stride) add(EM[j]);
  U128 acc[OBS_Q];
  acc[0] = {(unsigned long long)sE, sE < 0 ? ~0ull : 0ull};  // sign-extended
  acc[1] = {sE2, 0ull};
  acc[2] = {sA, 0ull};
  acc[3] = {sM2, 0ull};
  acc[4] = sM4;
  __shared__ U128 s_part[OBS_THREADS / 32][OBS_Q];
  __shared__ int s_emin[OBS_THREADS / 32], s_emax[OBS_THREADS / 32];
  __shared__ bool s_last;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
  for (int q = 0; q < OBS_Q; ++q) {
    const U128 v = warp_sum_u128(acc[q]);
    if (lane == 0) s_part[warp][q] = v;
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    emin = min(emin, __shfl_xor_sync(0xffffffffu, emin, o));
    emax = max(emax, __shfl_xor_sync(0xffffffffu, emax, o));
  }
  if (lane == 0) {
    s_emin[warp] = emin;
    s_emax[warp] = emax;
  }
  __syncthreads();
  if (threadIdx.x < OBS_Q) {
    U128 t = {0ull, 0ull};
    for (int w = 0; w < OBS_THREADS / 32; ++w) u128_add(t, s_part[w][threadIdx.x].lo, s_part[w][threadIdx.x].hi);
    partial[(size_t)blockIdx.x * 12 + 2 * threadIdx.x] = t.lo;
    partial[(size_t)blockIdx.x * 12 + 2 * threadIdx.x + 1] = t.hi;
  }
  if (threadIdx.x == OBS_Q) {
    int lo = s_emin[0], hi = s_emax[0];
    for (int w = 1; w < OBS_THREADS / 32; ++w) {
      lo = min(lo, s_emin[w]);
      hi = max(hi, s_emax[w]);
    }
    partial[(size_t)blockIdx.x * 12 + 10] = (unsigned long long)(long long)lo;
    partial[(size_t)blockIdx.x * 12 + 11] = (unsigned long long)(long long)hi;
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    __threadfence();
    const unsigned done = atomicAdd(&st->obs_done, 1u);
    s_last = (done == gridDim.x - 1);
  }
  __syncthreads();
  if (!s_last) return;
  __threadfence();
  // final reduction by the last block: warp q < 5 adds the partials of sum q (lanes stride over the blocks, then a
  // warp tree; integer sums, so the order does not matter), warp 5 takes min / max of E
  __shared__ long long s_lohi[2];
  if (warp < OBS_Q) {
    U128 t = {0ull, 0ull};
    for (unsigned b = lane; b < gridDim.x; b += 32)
      u128_add(t, __ldcg(&partial[(size_t)b * 12 + 2 * warp]), __ldcg(&partial[(size_t)b * 12 + 2 * warp + 1]));
    t = warp_sum_u128(t);
    if (lane == 0) {
      st->obs[2 * warp] = t.lo;
      st->obs[2 * warp + 1] = t.hi;
    }
  } else if (warp == OBS_Q) {
    long long lo = 0x7fffffff, hi = -0x7fffffff;
    for (unsigned b = lane; b < gridDim.x; b += 32) {
      const long long l = (long long)__ldcg(&partial[(size_t)b * 12 + 10]), h = (long long)__ldcg(&partial[(size_t)b * 12 + 11]);
      lo = l < lo ? l : lo;
      hi = h > hi ? h : hi;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      const long long l = __shfl_xor_sync(0xffffffffu, lo, o), h = __shfl_xor_sync(0xffffffffu, hi, o);
      lo = l < lo ? l : lo;
      hi = h > hi ? h : hi;
    }
    if (lane == 0) {
      s_lohi[0] = lo;
      s_lohi[1] = hi;
    }
  }
  __syncthreads();
  if (mode == 0) {  // a5: partition table of the new population + the paper's diagnostics, before the commit flips `cur`
    balance_tile(st, off, part0, part1, part_stats, ba);
    __syncthreads();
  }
  if (threadIdx.x == 0) {
    long long lo = s_lohi[0], hi = s_lohi[1];
    if (lo > hi) lo = hi = -2 * N;  // empty population: cannot happen (R >= 1), keep the window valid
    st->lev_lo = (int)((lo + 2 * N) >> 2);
    st->lev_hi = (int)((hi + 2 * N) >> 2);
    st->obs_R = count;
    if (mode != 1) {  // commit: the new population becomes the current one
      st->R_parents = st->R;
      st->R = st->Rnew;
      st->replica_steps += st->Rnew;
      if (mode == 0) st->cur ^= 1u;
      st->slot0 = st->slot0_new;
      st->step += 1u;
      st->sum_lnQ += st->lnQ;
      st->Q_committed = st->Q;
      st->beta = sp->beta_next;
      if (sp->theta > 0) {
        st->T4 = sp->T4;
        st->T8 = sp->T8;
      }
    }
  }
}

// ---------------------------------------------------------------------------------------------------
// Order parameter of the spin glass (D1, reading G28): overlap q = sum_i sigma_i^a sigma_i^b =
// N - 2 popc(a xor b) of replica j and replica j + floor(R/2), histogram hist[(q + N) / 2] over j < floor(R/2).
// One warp per pair, lanes stride over the words of the two lattices (coalesced 128-byte rows); block-level histogram in
// shared memory when it fits (N + 1 <= 4097 bins), global atomics otherwise.  HBM: the population is read once.
// ---------------------------------------------------------------------------------------------------
constexpr int OVL_THREADS = 256;
constexpr int OVL_SMEM_BINS = 4097;
__global__ void __launch_bounds__(OVL_THREADS)
k_overlap_hist(const DevState* __restrict__ st, const uint32_t* __restrict__ spins0, const uint32_t* __restrict__ spins1,
               unsigned long long* __restrict__ hist, const int N) {
  __shared__ unsigned s_hist[OVL_SMEM_BINS];
  const bool use_smem = N + 1 <= OVL_SMEM_BINS;
  if (use_smem)
    for (int i = threadIdx.x; i <= N; i += OVL_THREADS) s_hist[i] = 0u;
  __syncthreads();
  const uint32_t* __restrict__ spins = st->cur ? spins1 : spins0;
  const unsigned long long half = st->R / 2ull;
  const int wrep = N / 32, lane = threadIdx.x & 31;
  const unsigned long long warps = (unsigned long long)gridDim.x * (OVL_THREADS / 32);
  for (unsigned long long j = (unsigned long long)blockIdx.x * (OVL_THREADS / 32) + (threadIdx.x >> 5); j < half; j += warps) {
    const uint32_t* a = spins + j * wrep;
    const uint32_t* b = spins + (j + half) * wrep;
    int diff = 0;
    if ((wrep & 127) == 0) {  // L >= 64: 128-bit loads, a warp covers 512 bytes of each lattice per step
      const uint4* a4 = reinterpret_cast<const uint4*>(a);
      const uint4* b4 = reinterpret_cast<const uint4*>(b);
      for (int w = lane; w < wrep / 4; w += 32) {
        const uint4 x = __ldg(a4 + w), y = __ldg(b4 + w);
        diff += __popc(x.x ^ y.x) + __popc(x.y ^ y.y) + __popc(x.z ^ y.z) + __popc(x.w ^ y.w);
      }
    } else {
      for (int w = lane; w < wrep; w += 32) diff += __popc(__ldg(a + w) ^ __ldg(b + w));
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) diff += __shfl_xor_sync(0xffffffffu, diff, o);
    if (lane == 0) {
      const int bin = N - diff;  // (q + N) / 2 with q = N - 2 diff
      if (use_smem) atomicAdd(&s_hist[bin], 1u);
      else atomicAdd(&hist[bin], 1ull);
    }
  }
  __syncthreads();
  if (use_smem)
    for (int i = threadIdx.x; i <= N; i += OVL_THREADS)
      if (s_hist[i]) atomicAdd(&hist[i], (unsigned long long)s_hist[i]);
}

// ---------------------------------------------------------------------------------------------------
// Adaptive temperature step (PAPER.md:108 -> ref. [4]; A9, reading G25): the largest dbeta in (0, dbeta_max]
// whose histogram overlap alpha(dbeta) = (1/R) sum_j min(1, tau_j(dbeta)) is >= target.  tau_j depends on j only through
// the energy level, so one pass builds the level histogram of the population (k_level_hist) and one block bisects on it
// (k_adaptive_step): 40 halvings, each two block reductions over the occupied levels.
// ---------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(OBS_THREADS)
k_level_hist(const DevState* __restrict__ st, const int32_t* __restrict__ EM0, const int32_t* __restrict__ EM1,
             unsigned* __restrict__ hist, const int N) {
  const int32_t* __restrict__ E = st->cur ? EM1 : EM0;
  const unsigned long long R = st->R;
  const unsigned long long stride = (unsigned long long)gridDim.x * OBS_THREADS;
  for (unsigned long long j = (unsigned long long)blockIdx.x * OBS_THREADS + threadIdx.x; j < R; j += stride)
    atomicAdd(&hist[em_level(E[j], N)], 1u);
}

__device__ __forceinline__ double block_sum_256(double v, double* s_red) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  __syncthreads();  // s_red of the previous call has been consumed
  if ((threadIdx.x & 31) == 0) s_red[threadIdx.x >> 5] = v;
  __syncthreads();
  double t = 0.0;
#pragma unroll
  for (int w = 0; w < OBS_THREADS / 32; ++w) t += s_red[w];
  return t;
}

__global__ void __launch_bounds__(OBS_THREADS)
k_adaptive_step(DevState* st, unsigned* __restrict__ hist, const int N, const double target, const double dbeta_max,
                const int iters) {
  __shared__ double s_red[OBS_THREADS / 32];
  const int lev_lo = st->lev_lo, lev_hi = st->lev_hi;
  const double R = (double)st->R;
  const int e_off = st->e_off;
  auto overlap = [&](double dbeta) {
    double sw = 0.0;
    for (int lev = lev_lo + threadIdx.x; lev <= lev_hi; lev += OBS_THREADS)
      sw += (double)hist[lev] * exp(-dbeta * (double)(4 * lev - 2 * N + e_off));
    const double Q = block_sum_256(sw, s_red) / R;
    double sa = 0.0;
    for (int lev = lev_lo + threadIdx.x; lev <= lev_hi; lev += OBS_THREADS) {
      const double tau = exp(-dbeta * (double)(4 * lev - 2 * N + e_off)) / Q;
      sa += (double)hist[lev] * (tau < 1.0 ? tau : 1.0);
    }
    return block_sum_256(sa, s_red) / R;
  };
  double result = dbeta_max;
  if (!(overlap(dbeta_max) >= target)) {
    double lo = 0.0, hi = dbeta_max;  // alpha(lo) >= target > alpha(hi)
    for (int it = 0; it < iters; ++it) {
      const double mid = 0.5 * (lo + hi);
      if (overlap(mid) >= target) lo = mid;  // block-uniform: every thread holds the same sums
      else hi = mid;
    }
    result = lo;
  }
  __syncthreads();
  for (int lev = lev_lo + threadIdx.x; lev <= lev_hi; lev += OBS_THREADS) hist[lev] = 0u;  // ready for the next call
  if (threadIdx.x == 0) st->adaptive_dbeta = result;
}

}  // namespace pa
