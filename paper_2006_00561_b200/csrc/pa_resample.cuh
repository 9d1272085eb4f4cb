// pa_resample.cuh -- a1..a6: reweighting (eq. 3, 4), Poisson copy counts, single-pass exclusive scan,
// partition balance and the replica gather-copy.  PAPER.md:44-56, :84, :94, :104-106; C5, A4, A5, A6.
//
// lambda_j depends on j only through the integer energy E_j = 4*lev - 2N, lev = 0..N, so everything that is
// floating point is tabulated per energy LEVEL; the per-replica kernels only look the tables up.  A population
// occupies a few hundred adjacent levels [lev_lo, lev_hi] (recorded by k_observe when the population is written), so
// the tables are built for that window only (w inside k_q_reduce, the rest by k_levels_tau) and their hot part is held
// in shared memory.  The arithmetic per level is exactly the sequence written in DESIGN.md.
#pragma once
#include <type_traits>

#include "pa_common.cuh"

namespace pa {

constexpr int PO_KMAX = 64;            // A4: cap of the CDF inversion loop
constexpr int PO_ROW = 72;             // F_0 .. F_64 per level, padded to 72 doubles (64-byte aligned rows)
constexpr unsigned M_OVERFLOW = 0xffffffffu;

struct LevelTables {
  double* tau;      // [N+1]  w / Q
  double* mu;       // [N+1]  lambda / m
  uint32_t* m;      // [N+1]  number of chunks (0: lambda <= 0; M_OVERFLOW: lambda >= 2^31)
  double* cdf;      // [N+1][65]  F_k of Poisson(mu) built by the A4 recurrence
};

// w_e = exp(-dbeta * e) of energy level lev (e = 4 lev - 2N + e_off; e_off = 0 unless a +-J sample has an odd number of
// negative bonds, pa_common.cuh): the ONE expression that k_q_reduce (eq. 3) and
// k_levels_tau (eq. 4) both evaluate, so that tau = w / Q uses the very bits that were summed into Q
__device__ __forceinline__ double level_weight(double dbeta, int lev, int N, int e_off) {
  const double e = (double)(4 * lev - 2 * N + e_off);
  return exp(-dbeta * e);
}

// ---------------------------------------------------------------------------------------------------
// level_tables: per level tau = w / Q (eq. 4), lambda = tau * scale, and the A4 chunk tables
// (m, mu, F_0..F_64).  Only individually rounded IEEE operations (no FMA contraction).  Run by the last block of
// k_q_reduce, one thread per occupied level (a few hundred levels, up to 64 dependent divisions each).
// ---------------------------------------------------------------------------------------------------
__device__ __forceinline__ double expneg_a4(double mu) {
  // c_i = nearest double to (-1)^i / i!, i = 0..14
  constexpr double c[15] = {0x1.0000000000000p+0,   -0x1.0000000000000p+0,  0x1.0000000000000p-1,
                            -0x1.5555555555555p-3,  0x1.5555555555555p-5,   -0x1.1111111111111p-7,
                            0x1.6c16c16c16c17p-10,  -0x1.a01a01a01a01ap-13, 0x1.a01a01a01a01ap-16,
                            -0x1.71de3a556c734p-19, 0x1.27e4fb7789f5cp-22,  -0x1.ae64567f544e4p-26,
                            0x1.1eed8eff8d898p-29,  -0x1.6124613a86d09p-33, 0x1.93974a8c07c9dp-37};
  const double t = __dmul_rn(mu, 0.0625);
  double p = c[14];
#pragma unroll
  for (int i = 13; i >= 0; --i) p = __dadd_rn(__dmul_rn(p, t), c[i]);
#pragma unroll
  for (int s = 0; s < 4; ++s) p = __dmul_rn(p, p);
  return p;
}

__device__ __forceinline__ void level_tables(double dbeta, int lev, int N, int e_off, double Q, double scale, const LevelTables& tb,
                                             const int rule /* 0 Poisson, 1 nearest (A4b), 2 systematic (A4c) */) {
  const double tau = __ddiv_rn(level_weight(dbeta, lev, N, e_off), Q);
  const double lambda = __dmul_rn(tau, scale);
  tb.tau[lev] = tau;
  double* F = tb.cdf + (size_t)lev * PO_ROW;
  if (!(lambda > 0.0)) {
    tb.m[lev] = 0u;
    tb.mu[lev] = 0.0;
    return;
  }
  if (!(lambda < 2147483648.0)) {  // would exceed any capacity: reported as PA_ECAPACITY if a replica sits here
    tb.m[lev] = M_OVERFLOW;
    tb.mu[lev] = 0.0;
    return;
  }
  if (rule == 2) {  // A4c: Lam = floor(lambda * 2^32) as a 64-bit integer (exact), kept in the mu slot
    tb.m[lev] = 1u;
    tb.mu[lev] = __longlong_as_double((long long)floor(__dmul_rn(lambda, 4294967296.0)));
    F[0] = 2.0; F[1] = 2.0; F[2] = 2.0; F[3] = 2.0;
    return;
  }
  if (rule == 1) {  // A4b: n = floor(lambda) + [u > 1 - frac(lambda)]: one uniform per parent, never a heavy parent
    const double fl = floor(lambda);
    tb.m[lev] = 1u;
    tb.mu[lev] = lambda;
    F[0] = __dsub_rn(1.0, __dsub_rn(lambda, fl));              // threshold
    F[1] = __longlong_as_double((long long)fl);                // floor(lambda) as an integer bit pattern
    F[2] = 2.0;
    F[3] = 2.0;
    return;
  }
  long long m = (long long)ceil(__ddiv_rn(lambda, 8.0));
  if (m < 1) m = 1;
  const double mu = __ddiv_rn(lambda, (double)m);
  tb.m[lev] = (unsigned)m;
  tb.mu[lev] = mu;
  double p = expneg_a4(mu), Fk = p;
  F[0] = Fk;
  int k = 1;
  for (; k <= PO_KMAX; ++k) {
    p = __ddiv_rn(__dmul_rn(p, mu), (double)k);
    const double Fn = __dadd_rn(Fk, p);
    F[k] = Fn;
    // past the mode (k > mu) p only shrinks: once it no longer moves F, no later term does (identical bits, fewer
    // dependent divisions)
    if (Fn == Fk && (double)k > mu) break;
    Fk = Fn;
  }
  for (++k; k <= PO_KMAX; ++k) F[k] = Fk;
}

// ---------------------------------------------------------------------------------------------------
// k_q_reduce: eq. 3, first kernel of every step (it also resets the per-step counters and the scan's tile
// descriptors).  The population occupies the levels lev_lo..lev_hi (found by k_observe when the population was
// written); every block tabulates w for that window in shared memory (a few hundred exp per block), then: grid-stride
// 128-bit loads of E, look-up, per-thread serial sum, warp-shuffle tree, block partials; the last block to finish adds
// the partials in index order (deterministic for a given grid) and writes sumw, Q = sumw / R, ln Q, scale = R0 / R,
// and then the per-level tables of eq. 4 and of the Poisson sampler (level_tables above).
// A window wider than QW_MAX levels (crafted test populations) evaluates exp per replica instead: same bits.
// ---------------------------------------------------------------------------------------------------
constexpr int RED_THREADS = 256;
#ifndef PA_RED_UNR8
#define PA_RED_UNR8 0
#endif
constexpr int QW_MAX = 2048;

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

__global__ void __launch_bounds__(RED_THREADS)
k_q_reduce(DevState* st, const StepParams* __restrict__ sp, const int32_t* __restrict__ EM0,
           const int32_t* __restrict__ EM1, int N, double* __restrict__ partial, double R0,
           unsigned long long* __restrict__ tile_desc, int n_desc, LevelTables tb, int nearest) {
  grid_dependency_wait();
  const unsigned long long tid = (unsigned long long)blockIdx.x * RED_THREADS + threadIdx.x;
  const unsigned long long stride = (unsigned long long)gridDim.x * RED_THREADS;
  if (tid == 0) {  // counters of the later kernels of this step (reduce_done is reset by the last block below)
    st->scan_tile = 0u;
    st->scan_overflow = 0u;
    st->obs_done = 0u;
  }
  for (unsigned long long i = tid; i < (unsigned long long)n_desc; i += stride) tile_desc[i] = 0ull;
  if (st->status != ST_OK) return;
  const int32_t* __restrict__ E = st->cur ? EM1 : EM0;  // packed E/4 : M/2 words (pa_common.cuh)
  const unsigned long long R = st->R;
  const double dbeta = sp->dbeta;
  const int lev_lo = st->lev_lo, W = st->lev_hi - lev_lo + 1;
  const int halfN = N >> 1, e_off = st->e_off;
  const unsigned long long nvec = R / 4;
  const int4* __restrict__ E4 = reinterpret_cast<const int4*>(E);  // the buffers are 256-byte aligned
  __shared__ double s_w[QW_MAX];
  double acc = 0.0;
  if (W <= QW_MAX) {
    for (int i = threadIdx.x; i < W; i += RED_THREADS) s_w[i] = level_weight(dbeta, lev_lo + i, N, e_off);
    __syncthreads();
    const int shift = halfN - lev_lo;  // level - lev_lo = E / 4 + N / 2 - lev_lo
    auto wl = [&](int w) { return s_w[(w >> 16) + shift]; };
    unsigned long long v = tid;
#if PA_RED_UNR8
    for (; v + 7 * stride < nvec; v += 8 * stride) {  // eight 128-bit loads in flight per thread
      int4 x[8];
#pragma unroll
      for (int u = 0; u < 8; ++u) x[u] = __ldg(E4 + v + u * stride);
      double t[8];
#pragma unroll
      for (int u = 0; u < 8; ++u) t[u] = (wl(x[u].x) + wl(x[u].y)) + (wl(x[u].z) + wl(x[u].w));
      acc += ((t[0] + t[1]) + (t[2] + t[3])) + ((t[4] + t[5]) + (t[6] + t[7]));
    }
#endif
    for (; v + 3 * stride < nvec; v += 4 * stride) {  // four 128-bit loads in flight per thread
      const int4 a = __ldg(E4 + v), b = __ldg(E4 + v + stride), c = __ldg(E4 + v + 2 * stride), d = __ldg(E4 + v + 3 * stride);
      acc += (((wl(a.x) + wl(a.y)) + (wl(a.z) + wl(a.w))) + ((wl(b.x) + wl(b.y)) + (wl(b.z) + wl(b.w)))) +
             (((wl(c.x) + wl(c.y)) + (wl(c.z) + wl(c.w))) + ((wl(d.x) + wl(d.y)) + (wl(d.z) + wl(d.w))));
    }
    for (; v < nvec; v += stride) {
      const int4 a = __ldg(E4 + v);
      acc += (wl(a.x) + wl(a.y)) + (wl(a.z) + wl(a.w));
    }
    for (unsigned long long j = 4 * nvec + tid; j < R; j += stride) acc += wl(E[j]);
  } else {
    auto wl = [&](int w) { return level_weight(dbeta, (w >> 16) + halfN, N, e_off); };
    unsigned long long v = tid;
    for (; v < nvec; v += stride) {
      const int4 a = __ldg(E4 + v);
      acc += (wl(a.x) + wl(a.y)) + (wl(a.z) + wl(a.w));
    }
    for (unsigned long long j = 4 * nvec + tid; j < R; j += stride) acc += wl(E[j]);
  }

  __shared__ double s_part[RED_THREADS / 32];
  __shared__ bool s_last;
  acc = warp_sum(acc);
  if ((threadIdx.x & 31) == 0) s_part[threadIdx.x >> 5] = acc;
  __syncthreads();
  if (threadIdx.x == 0) {
    double b = 0.0;
#pragma unroll
    for (int w = 0; w < RED_THREADS / 32; ++w) b += s_part[w];
    partial[blockIdx.x] = b;
    __threadfence();
    const unsigned done = atomicAdd(&st->reduce_done, 1u);
    s_last = (done == gridDim.x - 1);
  }
  __syncthreads();
  if (!s_last) return;
  __shared__ double s_Q;
  if (threadIdx.x < 32) {
    __threadfence();
    double t = 0.0;
    for (unsigned b = threadIdx.x; b < gridDim.x; b += 32) t += __ldcg(&partial[b]);
    t = warp_sum(t);
    if (threadIdx.x == 0 && st->dist) {  // a shard: Q needs every rank's sum (k_dist_tables finishes the job)
      st->sumw = t;
      st->reduce_done = 0u;
    }
    if (threadIdx.x == 0 && !st->dist) {
      const double Q = t / (double)R;
      st->sumw = t;
      st->Q = Q;
      st->lnQ = log(Q);
      st->scale = R0 / (double)R;
      st->reduce_done = 0u;  // every block has arrived: ready for the next step
      s_Q = Q;
    }
  }
  __syncthreads();
  if (st->dist) return;
  // a2 per level: the tables of the occupied window (only that window is ever looked up)
  {
    const double Q = s_Q, scale = R0 / (double)R;
    const int lev_hi = st->lev_hi < N ? st->lev_hi : N;
    for (int lev = lev_lo + threadIdx.x; lev <= lev_hi; lev += RED_THREADS) level_tables(dbeta, lev, N, e_off, Q, scale, tb, nearest);
  }
}

// ---------------------------------------------------------------------------------------------------
// k_dist_tables: multi-GPU shard.  Every rank has summed its own weights (k_q_reduce); the host has added the ranks'
// sums in rank order (sumw_global, R_global).  One block: Q = sumw / R over the WHOLE population (the
// central node "sends this number to the nodes as the normalization factor"), ln Q, scale = R0 / R, and the level
// tables of this rank's occupied window.
// ---------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(RED_THREADS)
k_dist_tables(DevState* st, const StepParams* __restrict__ sp, int N, double sumw_global, double R_global, double R0,
              LevelTables tb, int nearest) {
  grid_dependency_wait();
  if (st->status != ST_OK) return;
  const double Q = sumw_global / R_global, scale = R0 / R_global;
  if (threadIdx.x == 0) {
    st->Q = Q;
    st->lnQ = log(Q);
    st->scale = scale;
  }
  const int lev_hi = st->lev_hi < N ? st->lev_hi : N;
  for (int lev = st->lev_lo + threadIdx.x; lev <= lev_hi; lev += RED_THREADS) level_tables(sp->dbeta, lev, N, st->e_off, Q, scale, tb, nearest);
}

// ---------------------------------------------------------------------------------------------------
// k_poisson_scan: a2-a4.  n_j ~ Poisson(lambda_j) by chunked CDF inversion with keyed uniforms, fused with a
// single-pass exclusive scan (decoupled look-back).  Tile = 256 threads x 8 parents = 2048 parents.
//   phase 1  every parent with m >= 1 draws its chunk 0 (one Philox block per parent, 8 parents per thread);
//   phase 2  the remaining chunks (c = 1 .. m-1) of the tile's heavy parents (lambda > 8; 2 % of the parents but
//            60 % of the children in config 5) form ONE flat work list that all 256 threads share, so that a parent
//            with lambda = 10^4 (1250 chunks) costs the tile 5 passes instead of serialising one warp; counts are
//            integer sums, so the result does not depend on who draws which chunk;
//   phase 3  block scan of the counts, look-back across tiles, offsets / counts written.  Then what the consumer of
//            the step needs to find the parents:
//            MAP (theta > 0)   the child -> parent map parent_of[i] (A5: the unique j with off_j <= i < off_j + n_j),
//                              expanded warp by warp: the 256 parents of a warp own one contiguous range of children,
//                              which the warp marks and max-scans 256 children at a time in its slice of shared memory
//                              (no block barrier, coalesced stores); the sweep's gather-on-load reads it;
//            !MAP (theta = 0)  only the parent that covers the first child of every copy tile; k_copy walks the
//                              offsets from there (measured on config 5: the full map costs the scan 0.05 ms and does
//                              not make the copy faster).
// ---------------------------------------------------------------------------------------------------
constexpr int SCAN_THREADS = 256;
constexpr int SCAN_ROUNDS = 8;
constexpr int SCAN_TILE = SCAN_THREADS * SCAN_ROUNDS;

constexpr unsigned long long DESC_AGG = 1ull << 62, DESC_PREFIX = 2ull << 62, DESC_VAL = (1ull << 62) - 1;

// u = ((x >> 12) + 0.5) * 2^-52 from the two keyed words of chunk c, built without an int->double conversion:
// 1 + k 2^-52 has the bits 0x3FF0... | k, and subtracting 1 - 2^-53 gives (2k + 1) 2^-53 exactly.
__device__ __forceinline__ double chunk_uniform(const uint4& w, unsigned odd) {
  const uint32_t hi = odd ? w.z : w.x, lo = odd ? w.w : w.y;
  const unsigned long long x = ((unsigned long long)hi << 32) | lo;
  return __longlong_as_double((long long)(0x3FF0000000000000ull | (x >> 12))) - 0x1.fffffffffffffp-1;
}
// k = #{i < 64 : u > F_i}.  F is non-decreasing (p_k >= 0), so this count equals the A4 loop
// "while (u > F && k < 64) ++k"; rows are 64-byte aligned, four entries per step.
__device__ __forceinline__ unsigned cdf_count4(const double2* __restrict__ F2, int g, double u) {
  const double2 a = __ldg(F2 + 2 * g), b = __ldg(F2 + 2 * g + 1);
  return (unsigned)(u > a.x) + (unsigned)(u > a.y) + (unsigned)(u > b.x) + (unsigned)(u > b.y);
}
__device__ __forceinline__ unsigned cdf_search_from(const double2* __restrict__ F2, int g0, double u) {
  unsigned k = 0;
#pragma unroll 1
  for (int g = g0; g < PO_KMAX / 4; ++g) {
    const unsigned c4 = cdf_count4(F2, g, u);
    k += c4;
    if (c4 < 4u) break;
  }
  return k;
}
__device__ __forceinline__ unsigned draw_chunk(const double* __restrict__ F, uint32_t j, unsigned long long c,
                                               uint32_t c3, const PhiloxKey& key) {
  const uint4 w = philox4x32_10((uint32_t)(c >> 1), j, 0u, c3, key);
  return cdf_search_from(reinterpret_cast<const double2*>(F), 0, chunk_uniform(w, (unsigned)(c & 1ull)));
}

struct ScanOut {
  uint32_t* off;            // [R + 1] exclusive offsets, off[R] = R'
  uint32_t* n;              // [R] copy counts (PA_KEEP_COUNTS) or null
  double* tau;              // [R] weights (PA_KEEP_TAU) or null
  unsigned long long* tile_desc;
  uint32_t* parent_of;      // MAP:  [R'] child -> parent map (theta > 0: read by the sweep's gather-on-load)
  uint32_t* tile_parent;    // !MAP: per copy tile the parent covering its first child (theta = 0: read by k_copy)
};

constexpr int SCAN_BATCH = 4;  // independent Philox chains in flight per thread
#ifndef PA_SCAN_HW
#define PA_SCAN_HW 192
#endif
constexpr int SCAN_HW = PA_SCAN_HW;
constexpr unsigned NO_TILE = 0xffffffffu;

// The kernel is software-pipelined over tiles: a block draws the counts of tile B and publishes its aggregate BEFORE it
// resolves the prefix of its previous tile A and writes A's offsets, so the look-back latency (descriptors of up to
// A tiles, 32 per round trip) is hidden behind B's sampling.  Every ticket holder publishes its aggregate before it
// waits on anything, so the look-back cannot deadlock.
#ifndef PA_SCAN_MINB
#define PA_SCAN_MINB 6
#endif
// RULE: 0 Poisson (A4), 1 nearest integers (A4b), 2 the copy counts are GIVEN in out.n (systematic resampling, A4c: written
// by k_sys_counts) and only scanned and placed here
template <bool KEEP, bool MAP, int RULE>
__global__ void __launch_bounds__(SCAN_THREADS, (MAP ? PA_SCAN_MINB - 1 : PA_SCAN_MINB))
k_poisson_scan(DevState* st, const int32_t* __restrict__ EM0, const int32_t* __restrict__ EM1, LevelTables tb, int N,
               ScanOut out, int copy_shift, unsigned long long capacity, const PhiloxKey key) {
  grid_dependency_wait();
  if (st->status != ST_OK) return;
  __shared__ unsigned s_tile;
  __shared__ unsigned s_flag;            // bit 0: a parent of this block sits on an overflowing level
  __shared__ unsigned long long s_pack;  // (total extra chunks << 12) | number of heavy parents   (one atomic sequence)
  __shared__ unsigned long long s_warp_tot[SCAN_THREADS / 32];
  __shared__ unsigned long long s_prefix;
  __shared__ __align__(16) unsigned s_cnt[2][SCAN_TILE];
  __shared__ uint32_t s_hstart[SCAN_TILE];  // first work-list position of heavy parent h (sum of lambda = R0 < 2^31: fits)
  __shared__ unsigned short s_hitem[SCAN_TILE];       // its item index inside the tile
  // the first CDF group F_0..F_3 and the chunk count m of the first SCAN_HW occupied levels, in shared memory: almost every
  // parent is decided by them (the population sits on a few hundred adjacent levels), the rest of a row stays in L1/L2
  __shared__ __align__(16) double s_head[SCAN_HW][4];
  __shared__ unsigned s_m[SCAN_HW];
  const int lev_lo = st->lev_lo;
  const bool all_cached = st->lev_hi - lev_lo < SCAN_HW;
  {
    const int W = min(st->lev_hi - lev_lo + 1, SCAN_HW);
    for (int i = threadIdx.x; i < 4 * W; i += SCAN_THREADS) s_head[i >> 2][i & 3] = tb.cdf[(size_t)(lev_lo + (i >> 2)) * PO_ROW + (i & 3)];
    for (int i = threadIdx.x; i < W; i += SCAN_THREADS) s_m[i] = tb.m[lev_lo + i];
  }
  const uint32_t R = (uint32_t)st->R;  // R <= capacity < 2^32 - 4096: parent indices fit 32 bits
  const unsigned ntiles = (R + SCAN_TILE - 1) / SCAN_TILE;
  const unsigned tile_end = ntiles;
  const int32_t* __restrict__ E = st->cur ? EM1 : EM0;  // packed E/4 : M/2 words
  const uint32_t c3 = ctr3(TAG_RESAMPLE, st->step + 1u);
  const uint32_t slot0 = st->slot0;  // the copy counts are keyed by the GLOBAL parent index (a multi-GPU shard: slot0 > 0)
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  if (threadIdx.x == 0) s_flag = 0u;
  unsigned prev = NO_TILE;
  int buf = 0;

  for (;;) {
    if (threadIdx.x == 0) {
      s_tile = atomicAdd(&st->scan_tile, 1u);
      s_pack = 0ull;
    }
    __syncthreads();
    const unsigned tile = s_tile < tile_end ? s_tile : NO_TILE;
    if (tile == NO_TILE && prev == NO_TILE) break;

    if (tile != NO_TILE) {
      const uint32_t tile_base = tile * SCAN_TILE;
      unsigned* cntb = s_cnt[buf];
      // phase 1: chunk 0 of every parent; item = r * 256 + tid (coalesced), SCAN_BATCH branch-free chains at a time.
      // Two instances of the batch: ALL = the whole occupied window is cached in shared memory (the usual case: no
      // global look-up and no address arithmetic for it on the common path), or the mixed path.
      auto batch = [&](auto all_tag, int r0) {
        constexpr bool ALL = decltype(all_tag)::value;
        uint32_t jj[SCAN_BATCH];
        int e[SCAN_BATCH];
        unsigned m[SCAN_BATCH], k[SCAN_BATCH], c4[SCAN_BATCH], hl[SCAN_BATCH];
        [[maybe_unused]] double u[SCAN_BATCH];
#pragma unroll
        for (int b = 0; b < SCAN_BATCH; ++b) {
          jj[b] = tile_base + (r0 + b) * SCAN_THREADS + threadIdx.x;
          e[b] = (jj[b] < R) ? __ldg(E + jj[b]) : (int)((uint32_t)(lev_lo - (N >> 1)) << 16);  // padding reads as the first occupied level
        }
#pragma unroll
        for (int b = 0; b < SCAN_BATCH; ++b) {
          const unsigned lev = (unsigned)em_level(e[b], N);
          hl[b] = lev - (unsigned)lev_lo;  // level relative to the cached window (>= SCAN_HW: not cached)
          const unsigned mm = (ALL || hl[b] < (unsigned)SCAN_HW) ? s_m[hl[b]] : __ldg(tb.m + lev);
          m[b] = (jj[b] < R) ? mm : 0u;
          if (KEEP) {
            if (out.tau && jj[b] < R) out.tau[jj[b]] = __ldg(tb.tau + lev);
          }
        }
        if constexpr (RULE != 2) {
#pragma unroll
          for (int b = 0; b < SCAN_BATCH; ++b) u[b] = chunk_uniform(philox4x32_10(0u, jj[b] + slot0, 0u, c3, key), 0u);
        }
#pragma unroll
        for (int b = 0; b < SCAN_BATCH; ++b) {  // rows of unused levels are masked below
          if constexpr (RULE == 2) {
            c4[b] = (jj[b] < R) ? __ldg(out.n + jj[b]) : 0u;
          } else if (ALL || hl[b] < (unsigned)SCAN_HW) {
            const double2 f01 = *reinterpret_cast<const double2*>(&s_head[hl[b]][0]);
            const double2 f23 = *reinterpret_cast<const double2*>(&s_head[hl[b]][2]);
            c4[b] = (unsigned)(u[b] > f01.x) + (unsigned)(u[b] > f01.y) + (unsigned)(u[b] > f23.x) + (unsigned)(u[b] > f23.y);
          } else {
            c4[b] = cdf_count4(reinterpret_cast<const double2*>(tb.cdf + (size_t)(hl[b] + (unsigned)lev_lo) * PO_ROW), 0, u[b]);
          }
        }
#pragma unroll
        for (int b = 0; b < SCAN_BATCH; ++b) {
          k[b] = c4[b];
          if constexpr (RULE == 2) {
            // given
          } else if constexpr (RULE == 1) {  // A4b: n = floor(lambda) + [u > 1 - frac(lambda)], both from the head of the row
            const double* F = (ALL || hl[b] < (unsigned)SCAN_HW) ? &s_head[hl[b]][0] : tb.cdf + (size_t)(hl[b] + (unsigned)lev_lo) * PO_ROW;
            k[b] = (unsigned)__double_as_longlong(F[1]) + (u[b] > F[0] ? 1u : 0u);
          } else if (c4[b] == 4u)
            k[b] += cdf_search_from(reinterpret_cast<const double2*>(tb.cdf + (size_t)(hl[b] + (unsigned)lev_lo) * PO_ROW), 1, u[b]);
          if (m[b] == M_OVERFLOW) {
            s_flag = 1u;
            m[b] = 0u;
          }
          if (m[b] == 0u) k[b] = 0u;
          if (m[b] > 1u) {
            const unsigned long long old = atomicAdd(&s_pack, ((unsigned long long)(m[b] - 1u) << 12) + 1ull);
            const unsigned h = (unsigned)(old & 0xfffull);
            s_hstart[h] = (uint32_t)(old >> 12);
            s_hitem[h] = (unsigned short)((r0 + b) * SCAN_THREADS + threadIdx.x);
          }
          cntb[(r0 + b) * SCAN_THREADS + threadIdx.x] = k[b];
        }
      };
      if (all_cached) {
#pragma unroll 1
        for (int r0 = 0; r0 < SCAN_ROUNDS; r0 += SCAN_BATCH) batch(std::true_type{}, r0);
      } else {
#pragma unroll 1
        for (int r0 = 0; r0 < SCAN_ROUNDS; r0 += SCAN_BATCH) batch(std::false_type{}, r0);
      }
      __syncthreads();
      // phase 2: flat work list over the extra chunks of the tile's heavy parents
      {
        const unsigned long long pack = s_pack;
        const unsigned long long W = pack >> 12;
        const unsigned nheavy = (unsigned)(pack & 0xfffull);  // <= SCAN_TILE = 2048 < 4096
        for (unsigned long long wk = threadIdx.x; wk < W; wk += SCAN_THREADS) {
          unsigned lo = 0, hi = nheavy;  // last h with s_hstart[h] <= wk
          while (hi - lo > 1u) {
            const unsigned mid = (lo + hi) >> 1;
            if (s_hstart[mid] <= wk) lo = mid; else hi = mid;
          }
          const unsigned item = s_hitem[lo];
          const uint32_t j = tile_base + item;
          const unsigned lev = (unsigned)em_level(__ldg(E + j), N);
          const unsigned kk = draw_chunk(tb.cdf + (size_t)lev * PO_ROW, j + slot0, 1ull + (wk - s_hstart[lo]), c3, key);
          if (kk) atomicAdd(&cntb[item], kk);
        }
      }
      __syncthreads();
      // aggregate of the tile, published at once
      {
        const uint4 a = *reinterpret_cast<const uint4*>(&cntb[SCAN_ROUNDS * threadIdx.x]);
        const uint4 b = *reinterpret_cast<const uint4*>(&cntb[SCAN_ROUNDS * threadIdx.x + 4]);
        unsigned long long t = (unsigned long long)a.x + a.y + a.z + a.w + b.x + b.y + b.z + b.w;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
        if (lane == 0) s_warp_tot[warp] = t;
        __syncthreads();
        if (threadIdx.x == 0) {
          unsigned long long tot = 0;
#pragma unroll
          for (int w = 0; w < SCAN_THREADS / 32; ++w) tot += s_warp_tot[w];
          atomicExch(&out.tile_desc[tile], (tile == 0 ? DESC_PREFIX : DESC_AGG) | tot);
        }
      }
    }

    if (prev != NO_TILE) {
      // phase 3 of the PREVIOUS tile: block scan (thread t owns the 8 consecutive items 8t .. 8t+7), look-back, outputs
      const unsigned* cntb = s_cnt[buf ^ 1];
      const uint32_t tile_base = prev * SCAN_TILE;
      unsigned cnt[SCAN_ROUNDS];
      {
        const uint4 a = *reinterpret_cast<const uint4*>(&cntb[SCAN_ROUNDS * threadIdx.x]);
        const uint4 b = *reinterpret_cast<const uint4*>(&cntb[SCAN_ROUNDS * threadIdx.x + 4]);
        cnt[0] = a.x; cnt[1] = a.y; cnt[2] = a.z; cnt[3] = a.w;
        cnt[4] = b.x; cnt[5] = b.y; cnt[6] = b.z; cnt[7] = b.w;
      }
      unsigned long long tsum = 0;
#pragma unroll
      for (int i = 0; i < SCAN_ROUNDS; ++i) tsum += cnt[i];
      unsigned long long inc = tsum;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const unsigned long long t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += t;
      }
      __syncthreads();  // s_warp_tot of the aggregate step above has been consumed
      if (lane == 31) s_warp_tot[warp] = inc;
      // decoupled look-back (warp 0); the aggregate of `prev` was published one iteration ago
      if (warp == 0) {
        unsigned long long prefix = 0;
        if (prev != 0u) {
          int look = (int)prev - 1;
          while (true) {
            const int idx = look - lane;
            unsigned long long d = DESC_PREFIX;  // lanes before tile 0 read as an empty prefix
            if (idx >= 0) {
              while (((d = *((volatile unsigned long long*)&out.tile_desc[idx])) >> 62) == 0ull) {}
            }
            const unsigned is_prefix = __ballot_sync(0xffffffffu, (d >> 62) == 2ull);
            unsigned long long v = d & DESC_VAL;
            if (is_prefix) {
              const int first = __ffs(is_prefix) - 1;  // nearest tile that already knows its inclusive prefix
              if (lane > first) v = 0ull;
            }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
            prefix += v;
            if (is_prefix) break;
            look -= 32;
          }
          if (lane == 0) {
            const unsigned long long own = *((volatile unsigned long long*)&out.tile_desc[prev]) & DESC_VAL;
            atomicExch(&out.tile_desc[prev], DESC_PREFIX | ((prefix + own) & DESC_VAL));
          }
        }
        if (lane == 0) s_prefix = prefix;
      }
      __syncthreads();
      unsigned long long warp_excl = 0, tile_total = 0;
#pragma unroll
      for (int w = 0; w < SCAN_THREADS / 32; ++w) {
        const unsigned long long t = s_warp_tot[w];
        if (w < warp) warp_excl += t;
        tile_total += t;
      }
      unsigned long long o64 = s_prefix + warp_excl + (inc - tsum);  // offset of the thread's first item

      // offsets and counts
      const uint32_t j0 = tile_base + SCAN_ROUNDS * threadIdx.x;
      const unsigned long long o_first = o64;
      uint32_t offs[SCAN_ROUNDS];
#pragma unroll
      for (int i = 0; i < SCAN_ROUNDS; ++i) {
        offs[i] = (uint32_t)o64;  // exact whenever R' fits the capacity
        if constexpr (!MAP) {  // for every copy tile the parent that covers its first child
          if (cnt[i] > 0u && j0 + i < R && o64 + cnt[i] <= capacity) {  // then o, o + cnt fit 32 bits
            const uint32_t o32 = (uint32_t)o64, ct1 = (1u << copy_shift) - 1u;
            const uint32_t t_first = (o32 + ct1) >> copy_shift, t_last = (o32 + cnt[i] - 1u) >> copy_shift;
#pragma unroll 1
            for (uint32_t t = t_first; t <= t_last; ++t) out.tile_parent[t] = j0 + i;
          }
        }
        o64 += cnt[i];
      }
      if (j0 + SCAN_ROUNDS <= R) {
        *reinterpret_cast<uint4*>(out.off + j0) = make_uint4(offs[0], offs[1], offs[2], offs[3]);
        *reinterpret_cast<uint4*>(out.off + j0 + 4) = make_uint4(offs[4], offs[5], offs[6], offs[7]);
        if (KEEP) {
          if (out.n) {
            *reinterpret_cast<uint4*>(out.n + j0) = make_uint4(cnt[0], cnt[1], cnt[2], cnt[3]);
            *reinterpret_cast<uint4*>(out.n + j0 + 4) = make_uint4(cnt[4], cnt[5], cnt[6], cnt[7]);
          }
        }
      } else {
#pragma unroll
        for (int i = 0; i < SCAN_ROUNDS; ++i) {
          if (j0 + i < R) {
            out.off[j0 + i] = offs[i];
            if (KEEP) {
              if (out.n) out.n[j0 + i] = cnt[i];
            }
          }
        }
      }
      // child -> parent map of the warp's 256 parents: their children are the contiguous range [w_lo, w_lo + w_n).  Chunks
      // of 256 children: every parent marks the position of its first child with its index inside the warp (+1), the
      // parent that reaches into the chunk from before it is the carry, an inclusive max-scan fills the rest.  A chunk
      // that lies inside one heavy parent's range is a plain fill.
      if constexpr (MAP) {
        unsigned* mk = const_cast<unsigned*>(cntb) + 256 * warp;  // the warp's slice: its counts are in registers by now
        const unsigned long long w_lo = __shfl_sync(0xffffffffu, o_first, 0);
        unsigned long long w_n64 = __shfl_sync(0xffffffffu, inc, 31);
        if (w_lo >= capacity) w_n64 = 0ull;  // a step that will not be committed: stay inside the buffers
        else if (w_lo + w_n64 > capacity) w_n64 = capacity - w_lo;
        const uint32_t w_n = (uint32_t)w_n64;  // <= capacity < 2^32
        const uint32_t wp_base = tile_base + 256u * (unsigned)warp;
        uint32_t* __restrict__ pw = out.parent_of + w_lo;
        // first child of each of the lane's parents relative to w_lo, saturated (counts of an uncommitted step may overflow)
        uint32_t fr[SCAN_ROUNDS + 1];
        {
          unsigned long long f = o_first - w_lo;
#pragma unroll
          for (int i = 0; i <= SCAN_ROUNDS; ++i) {
            fr[i] = f < 0xffffffffull ? (uint32_t)f : 0xffffffffu;
            if (i < SCAN_ROUNDS) f += cnt[i];
          }
        }
        __syncwarp();
        for (uint32_t c_lo = 0u; c_lo < w_n; c_lo += 256u) {
          // carry: the parent whose range starts before the chunk and reaches into it (at most one in the warp)
          unsigned carry = 0u, cover = 0u;
#pragma unroll
          for (int i = 0; i < SCAN_ROUNDS; ++i)
            if (fr[i] < c_lo && fr[i + 1] > c_lo) {
              carry = (unsigned)(SCAN_ROUNDS * lane + i + 1);
              cover = fr[i + 1] - c_lo;  // children of the chunk it covers (may exceed 256)
            }
          carry = __reduce_max_sync(0xffffffffu, carry);
          cover = __reduce_max_sync(0xffffffffu, cover);
          const unsigned n_here = w_n - c_lo < 256u ? w_n - c_lo : 256u;
          if (cover >= n_here) {  // warp-uniform: the whole chunk belongs to the carry parent
#pragma unroll
            for (int k = 0; k < 8; ++k) {
              const unsigned c = (unsigned)lane + 32u * k;
              if (c < n_here) pw[c_lo + c] = wp_base + carry - 1u;
            }
            continue;
          }
#pragma unroll
          for (int k = 0; k < 8; ++k) mk[lane + 32 * k] = 0u;
          __syncwarp();
#pragma unroll
          for (int i = 0; i < SCAN_ROUNDS; ++i)
            if (fr[i + 1] > fr[i] && fr[i] >= c_lo && fr[i] < c_lo + 256u) mk[fr[i] - c_lo] = (unsigned)(SCAN_ROUNDS * lane + i + 1);
          __syncwarp();
          uint4 a = *reinterpret_cast<const uint4*>(&mk[8 * lane]), b = *reinterpret_cast<const uint4*>(&mk[8 * lane + 4]);
          a.y = max(a.y, a.x); a.z = max(a.z, a.y); a.w = max(a.w, a.z);
          b.x = max(b.x, a.w); b.y = max(b.y, b.x); b.z = max(b.z, b.y); b.w = max(b.w, b.z);
          unsigned run = b.w;
#pragma unroll
          for (int o = 1; o < 32; o <<= 1) {
            const unsigned t = __shfl_up_sync(0xffffffffu, run, o);
            if (lane >= o) run = max(run, t);
          }
          unsigned before = __shfl_up_sync(0xffffffffu, run, 1);
          before = lane > 0 ? max(before, carry) : carry;
          a.x = max(a.x, before); a.y = max(a.y, before); a.z = max(a.z, before); a.w = max(a.w, before);
          b.x = max(b.x, before); b.y = max(b.y, before); b.z = max(b.z, before); b.w = max(b.w, before);
          *reinterpret_cast<uint4*>(&mk[8 * lane]) = a;
          *reinterpret_cast<uint4*>(&mk[8 * lane + 4]) = b;
          __syncwarp();
#pragma unroll
          for (int k = 0; k < 8; ++k) {
            const unsigned c = (unsigned)lane + 32u * k;
            if (c < n_here) pw[c_lo + c] = wp_base + mk[c] - 1u;
          }
          __syncwarp();
        }
      }
      if (threadIdx.x == 0) {
        if (prev == ntiles - 1) {
          const unsigned long long Rnew = s_prefix + tile_total;
          out.off[R] = (uint32_t)Rnew;
          st->Rnew = Rnew;
          const unsigned bad = Rnew > capacity ? (unsigned)ST_CAPACITY : (Rnew == 0ull ? (unsigned)ST_EXTINCT : (unsigned)ST_OK);
          if (bad != ST_OK) {
            atomicCAS(&st->status, (unsigned)ST_OK, bad);
            st->fail_step = st->step + 1u;
          }
        }
        if (s_flag & 1u) {  // a parent sits on a level with lambda >= 2^31: over any capacity (wins over "extinct")
          atomicExch(&st->status, (unsigned)ST_CAPACITY);
          st->fail_step = st->step + 1u;
        }
      }
    }
    if (tile == NO_TILE) break;
    prev = tile;
    buf ^= 1;
  }
}

// ---------------------------------------------------------------------------------------------------
// Systematic resampling (A4c): the copy counts come from the 64-bit prefix sum of Lam_j = floor(lambda_j 2^32),
// off_j = (C_j + U) >> 32.  Three small kernels in front of the scan, which then takes the counts as given:
//   k_sys_tile_sums   sum of Lam over every tile of 2048 parents
//   k_sys_scan_tiles  exclusive prefix over the tile sums (one block; the tiles are few: cap / 2048)
//   k_sys_counts      prefix inside the tile, n_j = ((C_j + Lam_j + U) >> 32) - ((C_j + U) >> 32)
// Integer arithmetic throughout: any order of the additions gives the oracle's bits.
// ---------------------------------------------------------------------------------------------------
constexpr int SYS_THREADS = 256, SYS_ITEMS = 8, SYS_TILE = SYS_THREADS * SYS_ITEMS;
static_assert(SYS_TILE == SCAN_TILE, "one tile geometry");

__device__ __forceinline__ unsigned long long sys_lam(const int32_t* __restrict__ E, uint32_t j, uint32_t R, const LevelTables& tb, int N) {
  if (j >= R) return 0ull;
  const int lev = em_level(__ldg(E + j), N);
  return __ldg(tb.m + lev) == 1u ? (unsigned long long)__double_as_longlong(__ldg(tb.mu + lev)) : 0ull;  // 0 / overflow levels: the scan reports them
}

__device__ __forceinline__ unsigned long long block_sum_u64(unsigned long long v, unsigned long long* s_w /* SYS_THREADS / 32 */) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  if ((threadIdx.x & 31) == 0) s_w[threadIdx.x >> 5] = v;
  __syncthreads();
  unsigned long long t = 0ull;
#pragma unroll
  for (int w = 0; w < SYS_THREADS / 32; ++w) t += s_w[w];
  return t;
}

__global__ void __launch_bounds__(SYS_THREADS)
k_sys_tile_sums(const DevState* __restrict__ st, const int32_t* __restrict__ EM0, const int32_t* __restrict__ EM1, LevelTables tb,
                int N, unsigned long long* __restrict__ tile_sum) {
  grid_dependency_wait();
  if (st->status != ST_OK) return;
  __shared__ unsigned long long s_w[SYS_THREADS / 32];
  const int32_t* __restrict__ E = st->cur ? EM1 : EM0;
  const uint32_t R = (uint32_t)st->R, base = blockIdx.x * SYS_TILE;
  unsigned long long v = 0ull;
  if (base < R) {
#pragma unroll
    for (int i = 0; i < SYS_ITEMS; ++i) v += sys_lam(E, base + i * SYS_THREADS + threadIdx.x, R, tb, N);
  }
  const unsigned long long t = block_sum_u64(v, s_w);
  if (threadIdx.x == 0) tile_sum[blockIdx.x] = t;
}

// in place: tile_sum[t] <- sum of the tiles before t
__global__ void __launch_bounds__(1024)
k_sys_scan_tiles(const DevState* __restrict__ st, unsigned long long* __restrict__ tile_sum, unsigned ntiles) {
  grid_dependency_wait();
  if (st->status != ST_OK) return;
  __shared__ unsigned long long s_w[32];
  __shared__ unsigned long long s_carry;
  if (threadIdx.x == 0) s_carry = 0ull;
  __syncthreads();
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  for (unsigned b = 0; b < ntiles; b += 1024u) {
    const unsigned t = b + threadIdx.x;
    const unsigned long long x = t < ntiles ? tile_sum[t] : 0ull;
    unsigned long long inc = x;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const unsigned long long y = __shfl_up_sync(0xffffffffu, inc, o);
      if (lane >= o) inc += y;
    }
    if (lane == 31) s_w[warp] = inc;
    __syncthreads();
    unsigned long long before = s_carry;
    for (int w = 0; w < warp; ++w) before += s_w[w];
    if (t < ntiles) tile_sum[t] = before + inc - x;
    __syncthreads();
    if (threadIdx.x == 1023) s_carry = before + inc;
    __syncthreads();
  }
}

__global__ void __launch_bounds__(SYS_THREADS)
k_sys_counts(const DevState* __restrict__ st, const int32_t* __restrict__ EM0, const int32_t* __restrict__ EM1, LevelTables tb, int N,
             const unsigned long long* __restrict__ tile_prefix, uint32_t* __restrict__ n_out, const PhiloxKey key) {
  grid_dependency_wait();
  if (st->status != ST_OK) return;
  __shared__ unsigned long long s_w[SYS_THREADS / 32];
  const int32_t* __restrict__ E = st->cur ? EM1 : EM0;
  const uint32_t R = (uint32_t)st->R, base = blockIdx.x * SYS_TILE;
  if (base >= R) return;
  const unsigned long long U = philox4x32_10(0u, 0u, 1u, ctr3(TAG_RESAMPLE, st->step + 1u), key).x;  // one uniform per step
  const uint32_t j0 = base + SYS_ITEMS * threadIdx.x;  // the thread's SYS_ITEMS consecutive parents
  unsigned long long lam[SYS_ITEMS], tsum = 0ull;
#pragma unroll
  for (int i = 0; i < SYS_ITEMS; ++i) {
    lam[i] = sys_lam(E, j0 + i, R, tb, N);
    tsum += lam[i];
  }
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  unsigned long long inc = tsum;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const unsigned long long y = __shfl_up_sync(0xffffffffu, inc, o);
    if (lane >= o) inc += y;
  }
  if (lane == 31) s_w[warp] = inc;
  __syncthreads();
  unsigned long long C = tile_prefix[blockIdx.x] + (inc - tsum);
  for (int w = 0; w < warp; ++w) C += s_w[w];
#pragma unroll
  for (int i = 0; i < SYS_ITEMS; ++i) {
    const unsigned long long before = (C + U) >> 32;
    C += lam[i];
    if (j0 + i < R) n_out[j0 + i] = (uint32_t)(((C + U) >> 32) - before);
  }
}

// ---------------------------------------------------------------------------------------------------
// k_copy: a6 for theta = 0 (with sweeps to follow, the sweep kernel gathers each child's lattice from its parent's slot
// through the child -> parent map that the scan then writes).  Child-centric gather.  Block t owns children
// [t*CT, (t+1)*CT): it starts from the parent that covers its first child (tile_parent, written by the scan), walks the offsets forward (coalesced), marks every
// parent at the position of its first child in shared memory and max-scans the marks into a child->parent map;
// then VT = S/16 lanes copy one lattice with 128-bit loads/stores.  Children are in parent order, so parent
// reads are monotone and repeated parents hit L1/L2.
// ---------------------------------------------------------------------------------------------------
constexpr int COPY_THREADS = 256;

template <int L>
struct CopyGeo {
  static constexpr int S = L * L / 8;                        // bytes per replica
  static constexpr int VB = S < 16 ? S : 16;                 // bytes per vector access
  static constexpr int VT = S / VB;                          // threads per child
  static constexpr int CT = S <= 128 ? 1024 : (S <= 512 ? 512 : 256);  // children per tile (multiple of COPY_THREADS)
  static_assert((CT & (CT - 1)) == 0, "k_poisson_scan divides child offsets by CT with a shift");
};

template <int VB> struct VecT;
template <> struct VecT<16> { using type = uint4; };
template <> struct VecT<8> { using type = uint2; };

template <int L>
__global__ void __launch_bounds__(COPY_THREADS)
k_copy(const DevState* __restrict__ st, const uint32_t* __restrict__ off, const uint32_t* __restrict__ tile_parent,
       uint32_t* spins0, uint32_t* spins1, int32_t* EM0, int32_t* EM1) {
  using CG = CopyGeo<L>;
  using V = typename VecT<CG::VB>::type;
  grid_dependency_wait();
  if (st->status != ST_OK) return;
  const unsigned long long R = st->R, Rnew = st->Rnew;
  const unsigned long long lim = R;  // off[0 .. R] are all in memory
  const unsigned long long i0 = (unsigned long long)blockIdx.x * CG::CT;
  if (i0 >= Rnew) return;
  const unsigned cur = st->cur;  // source = buffer cur, destination = buffer cur^1 (never the same memory)
  const V* __restrict__ src = reinterpret_cast<const V*>(cur ? spins1 : spins0);
  V* __restrict__ dst = reinterpret_cast<V*>(cur ? spins0 : spins1);
  const int32_t* __restrict__ EMs = cur ? EM1 : EM0;  // packed E/4 : M/2 words: one gather, one store per child
  int32_t* __restrict__ EMd = cur ? EM0 : EM1;
  const unsigned nchild = (unsigned)((Rnew - i0 < (unsigned long long)CG::CT) ? (Rnew - i0) : CG::CT);
  const unsigned long long i1 = i0 + nchild;

  __shared__ uint32_t s_par[CG::CT];
  __shared__ uint32_t s_wmax[COPY_THREADS / 32];
  for (int c = threadIdx.x; c < CG::CT; c += COPY_THREADS) s_par[c] = 0u;
  __syncthreads();
  const uint32_t j_first = tile_parent[blockIdx.x];
  if (threadIdx.x == 0) s_par[0] = j_first;
  // walk parents after j_first until their first child falls past the tile
  for (unsigned long long jb = (unsigned long long)j_first + 1;; jb += COPY_THREADS) {
    const unsigned long long j = jb + threadIdx.x;
    bool past = true;
    if (j < lim) {  // off[0 .. R] are all in memory: the scan kernel has finished
      const uint32_t o = off[j], o1 = off[j + 1];
      past = (o >= i1);
      if (!past && o1 > o) s_par[o - i0] = (uint32_t)j;  // o >= i0 because j > j_first
    }
    // off is monotone: once the first lane of a chunk is past, all later parents are
    if (__syncthreads_or(past && threadIdx.x == 0)) break;
  }
  __syncthreads();
  // inclusive max-scan of s_par (CT / COPY_THREADS consecutive entries per thread)
  {
    constexpr int PER = CG::CT / COPY_THREADS;
    uint32_t v[PER];
    uint32_t mx = 0u;
#pragma unroll
    for (int k = 0; k < PER; ++k) {
      mx = max(mx, s_par[threadIdx.x * PER + k]);
      v[k] = mx;
    }
    uint32_t inc = mx;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
      if (lane >= o) inc = max(inc, t);
    }
    if (lane == 31) s_wmax[warp] = inc;
    __syncthreads();
    uint32_t before = 0u;
    for (int w = 0; w < warp; ++w) before = max(before, s_wmax[w]);
    const uint32_t prev_lane = __shfl_up_sync(0xffffffffu, inc, 1);
    if (lane > 0) before = max(before, prev_lane);
#pragma unroll
    for (int k = 0; k < PER; ++k) s_par[threadIdx.x * PER + k] = max(v[k], before);
  }
  __syncthreads();

  // E, M of the children
  for (unsigned c = threadIdx.x; c < nchild; c += COPY_THREADS) {
    EMd[i0 + c] = EMs[s_par[c]];
  }
  // lattices: VT threads per child, 4 children in flight per thread group
  constexpr int GROUPS = COPY_THREADS / (CG::VT < COPY_THREADS ? CG::VT : COPY_THREADS);
  {
    const int sub = threadIdx.x % CG::VT, grp = threadIdx.x / CG::VT;
    constexpr int UNR = 4;
    unsigned c = grp;
    for (; c + (UNR - 1) * GROUPS < nchild; c += UNR * GROUPS) {
      V tmp[UNR];
#pragma unroll
      for (int u = 0; u < UNR; ++u) tmp[u] = src[(unsigned long long)s_par[c + u * GROUPS] * CG::VT + sub];
#pragma unroll
      for (int u = 0; u < UNR; ++u) dst[(i0 + c + u * GROUPS) * CG::VT + sub] = tmp[u];
    }
    for (; c < nchild; c += GROUPS) dst[(i0 + c) * CG::VT + sub] = src[(unsigned long long)s_par[c] * CG::VT + sub];
  }
}

}  // namespace pa
