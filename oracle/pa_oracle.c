/*
 * pa_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, scalar CPU statement of the population-annealing (PA) hot path of
 * arxiv 2006.00561 (Russkov, Chulkevich, Shchur), written from /root/reference/PAPER.md
 * and the readings listed in DESIGN.md ("Readings of the paper").  It exists so that
 * the CUDA path can be compared with something that a reader can check against the
 * paper by eye.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may load it.  It shares no code, header, table or constant
 * with paper_2006_00561_b200/csrc/ and neither side includes the other.
 *
 * Style rules kept here on purpose:
 *   - spins are handled as int8 values +1/-1 in a per-replica scratch array; the packed
 *     bit string is only the storage/interchange format and
 *     is converted bit by bit in unpack_replica()/pack_replica();
 *   - every loop is per site / per replica in the paper's order; no blocking, no bit tricks;
 *   - floating point is IEEE binary64, compiled with -ffp-contract=off (see build.py), sums
 *     are Neumaier-compensated;
 *   - OpenMP is used only across replicas (independent by construction) so that the timed
 *     CPU baseline can use the host's cores; results do not depend on the thread count.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): brute-force Z at L=4 against Kaufman's
 * closed form, density of states, PA ln Z against the exact finite-L value, closed forms
 * for Q/tau, Poisson moments/chi-square, expneg against exp, Philox against an independent
 * big-integer writing, zero-temperature and detailed-balance checks of the Metropolis
 * rule, global-flip covariance.  Section D1 (+-J spin glass, overlap histogram): tests/test_oracle_spin_glass.py --
 * numpy second writing on all 2^16 states of L = 4, parity law of E, gauge covariance onto the pinned ferromagnet,
 * hand-worked zero-temperature moves, Boltzmann chi-square and PA ln Z of a frustrated sample against enumeration.
 * Section A4c (systematic resampling): a Python-integer second writing with the big-integer Philox, floor / ceil and
 * population laws, E[n] = lambda.  Heating protocol (negative dbeta): ln Z of the 4x4 torus from its ground states.
 * No function here is "parity unpinned".
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* ------------------------------------------------------------------------------------------
 * Threads (only for the timed baseline; results are thread-count independent)
 * ---------------------------------------------------------------------------------------- */
int orc_max_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}
void orc_set_threads(int n) {
#ifdef _OPENMP
  if (n > 0) omp_set_num_threads(n);
#else
  (void)n;
#endif
}

/* ------------------------------------------------------------------------------------------
 * C3. Philox4x32-10 (Salmon et al., SC'11; not in the paper -- BASELINE.json north_star
 * asks for a counter-based Philox).  DESIGN.md "C3".
 * ---------------------------------------------------------------------------------------- */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
  uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
  uint32_t k0 = key[0], k1 = key[1];
  for (int round = 0; round < 10; ++round) {
    if (round > 0) { /* key schedule between rounds */
      k0 += 0x9E3779B9u;
      k1 += 0xBB67AE85u;
    }
    uint64_t p0 = (uint64_t)0xD2511F53u * (uint64_t)c0;
    uint64_t p1 = (uint64_t)0xCD9E8D57u * (uint64_t)c2;
    uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
    uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
    uint32_t n0 = hi1 ^ c1 ^ k0;
    uint32_t n1 = lo1;
    uint32_t n2 = hi0 ^ c3 ^ k1;
    uint32_t n3 = lo0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

enum { TAG_INIT = 0, TAG_RESAMPLE = 1, TAG_SWEEP = 2 };

static void philox_keyed(uint64_t seed, uint32_t c0, uint32_t c1, uint32_t c2, uint32_t tag,
                         uint32_t step, uint32_t w[4]) {
  uint32_t ctr[4] = {c0, c1, c2, (tag << 28) | step};
  uint32_t key[2] = {(uint32_t)(seed & 0xffffffffu), (uint32_t)(seed >> 32)};
  orc_philox4x32_10(ctr, key, w);
}

/* ------------------------------------------------------------------------------------------
 * C2. Bit layout: replica = N-bit little-endian string, bit b = y*L + x, word b>>5, bit b&31,
 * bit 1 <-> sigma = +1.  Storage only.
 * ---------------------------------------------------------------------------------------- */
static void unpack_replica(int L, const uint32_t* words, int8_t* s) {
  int N = L * L;
  for (int b = 0; b < N; ++b) s[b] = ((words[b >> 5] >> (b & 31)) & 1u) ? (int8_t)1 : (int8_t)-1;
}
static void pack_replica(int L, const int8_t* s, uint32_t* words) {
  int N = L * L;
  int nwords = (N + 31) / 32;
  for (int w = 0; w < nwords; ++w) words[w] = 0u;
  for (int b = 0; b < N; ++b)
    if (s[b] > 0) words[b >> 5] |= (1u << (b & 31));
}
/* words per replica: N/32 (N is a multiple of 32 for every supported L >= 8; for L = 4 and
 * L = 6 the last word is partly used and its unused bits are zero). */
int64_t orc_words_per_replica(int L) { return ((int64_t)L * L + 31) / 32; }

/* ------------------------------------------------------------------------------------------
 * C1. Energy, eq. (6):  H = -(J/2) sum' sigma sigma'  over all nearest neighbours
 * sigma' of every spin sigma, J = 1, periodic square lattice.  Magnetisation
 * M = sum sigma.
 * ---------------------------------------------------------------------------------------- */
static int32_t energy_of(int L, const int8_t* s) {
  int64_t twice = 0; /* sum over every spin of sigma * (its four neighbours) = 2 * sum over bonds */
  for (int y = 0; y < L; ++y)
    for (int x = 0; x < L; ++x) {
      int sig = s[y * L + x];
      int right = s[y * L + (x + 1) % L];
      int left = s[y * L + (x + L - 1) % L];
      int down = s[((y + 1) % L) * L + x];
      int up = s[((y + L - 1) % L) * L + x];
      twice += sig * (right + left + down + up);
    }
  return (int32_t)(-(twice / 2)); /* J/2 with J = 1; 'twice' is even */
}
static int32_t magnetisation_of(int L, const int8_t* s) {
  int32_t m = 0;
  for (int b = 0; b < L * L; ++b) m += s[b];
  return m;
}

void orc_energy_mag(int L, int64_t R, const uint32_t* packed, int32_t* E, int32_t* M) {
  int64_t wpr = orc_words_per_replica(L);
#pragma omp parallel
  {
    int8_t* s = (int8_t*)malloc((size_t)L * L);
#pragma omp for schedule(static)
    for (int64_t j = 0; j < R; ++j) {
      unpack_replica(L, packed + j * wpr, s);
      E[j] = energy_of(L, s);
      M[j] = magnetisation_of(L, s);
    }
    free(s);
  }
}

/* ------------------------------------------------------------------------------------------
 * D1. Second Hamiltonian behind the same step (PAPER.md:213 names the spin glass
 * as the complex system the method is meant for; reading G27): the 2D +-J Edwards-Anderson
 * model  H = - sum_<ij> J_ij sigma_i sigma_j  on the same periodic L x L lattice, one sample of
 * couplings J_ij = +-1 shared by all replicas.  Jx[y*L+x] couples (x,y)-(x+1,y), Jy[y*L+x] couples
 * (x,y)-(x,y+1), indices modulo L.  Every J = +1 is eq. (6).  E = 2u - 2N with u the number of
 * unsatisfied bonds; u keeps the parity of the number of negative bonds, so E = 2 (#negative) mod 4.
 * ---------------------------------------------------------------------------------------- */
static int32_t energy_of_J(int L, const int8_t* s, const int8_t* Jx, const int8_t* Jy) {
  int32_t e = 0; /* sum over the 2N bonds, each once: the bond to the right and the bond below every site */
  for (int y = 0; y < L; ++y)
    for (int x = 0; x < L; ++x) {
      int sig = s[y * L + x];
      e -= Jx[y * L + x] * sig * s[y * L + (x + 1) % L];
      e -= Jy[y * L + x] * sig * s[((y + 1) % L) * L + x];
    }
  return e;
}
void orc_energy_mag_J(int L, int64_t R, const uint32_t* packed, const int8_t* Jx, const int8_t* Jy, int32_t* E,
                      int32_t* M) {
  int64_t wpr = orc_words_per_replica(L);
#pragma omp parallel
  {
    int8_t* s = (int8_t*)malloc((size_t)L * L);
#pragma omp for schedule(static)
    for (int64_t j = 0; j < R; ++j) {
      unpack_replica(L, packed + j * wpr, s);
      E[j] = energy_of_J(L, s, Jx, Jy);
      M[j] = magnetisation_of(L, s);
    }
    free(s);
  }
}
int32_t orc_energy_int8_J(int L, const int8_t* s, const int8_t* Jx, const int8_t* Jy) { return energy_of_J(L, s, Jx, Jy); }

/* Order parameter of the spin glass ("the distribution of the order parameter for the spin-glass
 * model at each annealing step, averaging over the population"): overlap q_ab = sum_i sigma_i^a sigma_i^b of
 * replica a = j and replica b = j + floor(R/2), j = 0 .. floor(R/2)-1 (reading G28: partners half a population
 * apart, so that they are not siblings of one recent parent); hist[(q + N) / 2] counts the pairs (q = N mod 2). */
void orc_overlap_hist(int L, int64_t R, const uint32_t* packed, uint64_t* hist /* N+1 */) {
  int N = L * L;
  int64_t wpr = orc_words_per_replica(L), half = R / 2;
  int8_t* sa = (int8_t*)malloc((size_t)N);
  int8_t* sb = (int8_t*)malloc((size_t)N);
  for (int i = 0; i <= N; ++i) hist[i] = 0;
  for (int64_t j = 0; j < half; ++j) {
    unpack_replica(L, packed + j * wpr, sa);
    unpack_replica(L, packed + (j + half) * wpr, sb);
    int q = 0;
    for (int i = 0; i < N; ++i) q += sa[i] * sb[i];
    hist[(q + N) / 2] += 1;
  }
  free(sa);
  free(sb);
}

/* ------------------------------------------------------------------------------------------
 * A1. Initial population at beta0 = 0: every spin +1/-1 with equal probability.
 * C3 init keying: 32-bit word v of replica j <- w[v&3] of counter (v>>2, j, 0, tag0|0); spin b
 * is +1 iff bit (b&31) of word (b>>5) is set.
 * ---------------------------------------------------------------------------------------- */
void orc_init_population(int L, int64_t R, uint64_t seed, uint32_t* packed) {
  int N = L * L;
  int64_t wpr = orc_words_per_replica(L);
#pragma omp parallel
  {
    int8_t* s = (int8_t*)malloc((size_t)N);
#pragma omp for schedule(static)
    for (int64_t j = 0; j < R; ++j) {
      uint32_t w[4] = {0, 0, 0, 0};
      for (int b = 0; b < N; ++b) {
        uint32_t v = (uint32_t)(b >> 5); /* word that holds bit b */
        if ((b & 127) == 0)              /* one Philox block serves four consecutive words = 128 spins */
          philox_keyed(seed, v >> 2, (uint32_t)j, 0u, TAG_INIT, 0u, w);
        uint32_t word = w[v & 3];
        s[b] = ((word >> (b & 31)) & 1u) ? (int8_t)1 : (int8_t)-1;
      }
      pack_replica(L, s, packed + j * wpr);
    }
    free(s);
  }
}

/* ------------------------------------------------------------------------------------------
 * C5 / A2 / A3.  PAPER.md:46 eq. (3):  Q = sum_j exp[-(beta' - beta) E_j] / R  with R the
 * CURRENT population;  PAPER.md:51 eq. (4):  tau_j = exp[-(beta'-beta) E_j] / Q.
 * Neumaier-compensated sum.  orc_q_by_levels is the same sum grouped by energy level, kept as
 * a self-check (tests compare the two to 1e-14).
 * ---------------------------------------------------------------------------------------- */
double orc_q(int64_t R, const int32_t* E, double dbeta) {
  double sum = 0.0, comp = 0.0;
  for (int64_t j = 0; j < R; ++j) {
    double w = exp(-dbeta * (double)E[j]);
    double t = sum + w;
    if (fabs(sum) >= fabs(w)) comp += (sum - t) + w;
    else comp += (w - t) + sum;
    sum = t;
  }
  return (sum + comp) / (double)R;
}
double orc_q_by_levels(int64_t R, const int32_t* E, double dbeta, int N) {
  /* levels E = -2N, -2N+4, ..., 2N  (E = 0 mod 4, |E| <= 2N; C1) */
  int nlev = N + 1;
  int64_t* count = (int64_t*)calloc((size_t)nlev, sizeof(int64_t));
  for (int64_t j = 0; j < R; ++j) count[(E[j] + 2 * N) / 4] += 1;
  double sum = 0.0, comp = 0.0;
  for (int l = 0; l < nlev; ++l) {
    if (!count[l]) continue;
    double w = (double)count[l] * exp(-dbeta * (double)(4 * l - 2 * N));
    double t = sum + w;
    if (fabs(sum) >= fabs(w)) comp += (sum - t) + w;
    else comp += (w - t) + sum;
    sum = t;
  }
  free(count);
  return (sum + comp) / (double)R;
}
void orc_tau(int64_t R, const int32_t* E, double dbeta, double Q, double* tau) {
  for (int64_t j = 0; j < R; ++j) tau[j] = exp(-dbeta * (double)E[j]) / Q;
}

/* ------------------------------------------------------------------------------------------
 * A4.  Poisson copy counts, PAPER.md:54 ("We choose the number of replicas in the configuration
 * j from the Poisson distribution keeping the number of replicas close to the original one"):
 * n_j ~ Poisson(lambda_j), lambda_j = tau_j * (R0 / R)  (reading G2).
 * Sampler (the parity contract): split lambda into m chunks of mean mu <= 8,
 * each drawn by CDF inversion with one keyed uniform; only individually rounded IEEE + - * /.
 * ---------------------------------------------------------------------------------------- */
#define PO_CH 8.0
#define PO_KMAX 64
#define PO_DEG 14

/* exp(-mu) for 0 <= mu <= 8: degree-14 Taylor polynomial of exp(-t) at t = mu/16 (Horner),
 * then four squarings.  c_i = (-1)^i / i!  correctly rounded: i! <= 14! < 2^53 is exact in
 * binary64 and IEEE division rounds to nearest, so +-1.0/(double)i! IS the nearest double. */
double orc_expneg(double mu) {
  double c[PO_DEG + 1];
  double fact = 1.0;
  for (int i = 0; i <= PO_DEG; ++i) {
    if (i > 0) fact = fact * (double)i;
    c[i] = ((i & 1) ? -1.0 : 1.0) / fact;
  }
  double t = mu * 0.0625; /* 2^-4, exact scaling */
  double p = c[PO_DEG];
  for (int i = PO_DEG - 1; i >= 0; --i) p = (p * t) + c[i];
  for (int sq = 0; sq < 4; ++sq) p = p * p;
  return p;
}

/* uniform in (0,1) for chunk c of parent j (C3 resample keying): words (w[2(c&1)], w[2(c&1)+1])
 * of counter (c>>1, j, 0, tag1|step); x = (hi<<32)|lo; u = ((x>>12) + 0.5) * 2^-52 (exact). */
double orc_uniform_resample(uint64_t seed, uint32_t step, uint32_t j, uint64_t c) {
  uint32_t w[4];
  philox_keyed(seed, (uint32_t)(c >> 1), j, 0u, TAG_RESAMPLE, step, w);
  uint32_t hi = w[2 * (c & 1)], lo = w[2 * (c & 1) + 1];
  uint64_t x = ((uint64_t)hi << 32) | (uint64_t)lo;
  return ((double)(x >> 12) + 0.5) * 0x1p-52;
}

uint32_t orc_poisson(double lambda, uint64_t seed, uint32_t step, uint32_t j) {
  if (!(lambda > 0.0)) return 0u;
  int64_t m = (int64_t)ceil(lambda / PO_CH);
  if (m < 1) m = 1;
  double mu = lambda / (double)m;
  double p0 = orc_expneg(mu);
  uint64_t total = 0;
  for (int64_t c = 0; c < m; ++c) {
    double u = orc_uniform_resample(seed, step, j, (uint64_t)c);
    int k = 0;
    double p = p0, F = p0;
    while (u > F && k < PO_KMAX) {
      k += 1;
      p = (p * mu) / (double)k;
      F = F + p;
    }
    total += (uint64_t)k;
  }
  return (uint32_t)total;
}

void orc_poisson_counts(int64_t R, const double* tau, double scale, uint64_t seed, uint32_t step,
                        uint32_t* n) {
#pragma omp parallel for schedule(dynamic, 1024)
  for (int64_t j = 0; j < R; ++j) {
    double lambda = tau[j] * scale;
    n[j] = orc_poisson(lambda, seed, step, (uint32_t)j);
  }
}

/* ------------------------------------------------------------------------------------------
 * A4b.  Nearest-integer resampling, one of the "possible modifications of this step" the paper points to
 * (PAPER.md:54 -> ref. [3]; reading G24):  n_j = floor(lambda_j) + [u_j > 1 - frac(lambda_j)],
 * frac(lambda) = lambda - floor(lambda), u_j the keyed uniform of chunk 0 of parent j (the same number the Poisson
 * sampler would use).  E[n_j] = lambda_j like the Poisson rule, but n_j is one of the two integers next to lambda_j,
 * so the population size fluctuates much less.  floor, the subtractions and the comparison are exact / individually
 * rounded binary64 operations.
 * ---------------------------------------------------------------------------------------- */
uint32_t orc_nearest(double lambda, uint64_t seed, uint32_t step, uint32_t j) {
  if (!(lambda > 0.0)) return 0u;
  double fl = floor(lambda);
  double thr = 1.0 - (lambda - fl);
  double u = orc_uniform_resample(seed, step, j, 0u);
  return (uint32_t)fl + (u > thr ? 1u : 0u);
}
void orc_nearest_counts(int64_t R, const double* tau, double scale, uint64_t seed, uint32_t step, uint32_t* n) {
#pragma omp parallel for schedule(static)
  for (int64_t j = 0; j < R; ++j) n[j] = orc_nearest(tau[j] * scale, seed, step, (uint32_t)j);
}

/* ------------------------------------------------------------------------------------------
 * A4c.  Systematic resampling, another of the "possible modifications of this step" (PAPER.md:54 -> ref. [3]; DESIGN.md
 * reading G30): ONE keyed 32-bit uniform U per temperature step for the whole population, copy numbers from the
 * cumulative sum of the weights on a comb of spacing 1:
 *     Lam_j = floor(lambda_j * 2^32)  (exact: a power-of-two scaling and a floor of a binary64 number, 64-bit integer)
 *     C_j   = sum_{i<j} Lam_i         (exact 64-bit integer arithmetic: independent of the order of summation)
 *     off_j = (C_j + U) >> 32,   n_j = off_{j+1} - off_j,   R' = off_R
 * E[n_j] = Lam_j / 2^32 (= lambda_j up to 2^-32), n_j is one of the two integers next to it, and the population size
 * is floor(sum_j lambda_j) or that + 1: it stays at R0 instead of fluctuating like sqrt(R0).  U = word 0 of the Philox
 * counter (0, 0, 1, tag1|step): c2 = 1 keeps it apart from the per-parent chunk counters (c2 = 0).
 * ---------------------------------------------------------------------------------------- */
uint32_t orc_systematic_uniform(uint64_t seed, uint32_t step) {
  uint32_t w[4];
  philox_keyed(seed, 0u, 0u, 1u, TAG_RESAMPLE, step, w);
  return w[0];
}
void orc_systematic_counts(int64_t R, const double* tau, double scale, uint64_t seed, uint32_t step, uint32_t* n) {
  uint64_t U = orc_systematic_uniform(seed, step);
  uint64_t C = 0; /* running sum of Lam, sequential on purpose */
  for (int64_t j = 0; j < R; ++j) {
    double lambda = tau[j] * scale;
    uint64_t Lam = lambda > 0.0 ? (uint64_t)floor(lambda * 4294967296.0) : 0u;
    uint64_t before = (C + U) >> 32;
    C += Lam;
    n[j] = (uint32_t)(((C + U) >> 32) - before);
  }
}

/* ------------------------------------------------------------------------------------------
 * A9.  Adaptive temperature step ("Fluctuations can be made smaller and less frequent using the adaptive
 * temperature step, as discussed in the papers [4]"; reading G25).  The overlap of the energy histograms at
 * beta and beta + dbeta, estimated from the population as in ref. [4]:
 *     alpha(dbeta) = (1/R) sum_j min(1, tau_j(dbeta)),   tau_j by eq. 3-4,
 * is 1 at dbeta = 0 and decreases with dbeta.  The step is the largest dbeta in (0, dbeta_max] with
 * alpha(dbeta) >= target, located by `iters` bisection steps on [0, dbeta_max] (dbeta_max itself if it already
 * satisfies the target).
 * ---------------------------------------------------------------------------------------- */
double orc_overlap(int64_t R, const int32_t* E, double dbeta) {
  double Q = orc_q(R, E, dbeta);
  double sum = 0.0, comp = 0.0;
  for (int64_t j = 0; j < R; ++j) {
    double tau = exp(-dbeta * (double)E[j]) / Q;
    double w = tau < 1.0 ? tau : 1.0;
    double t = sum + w;
    if (fabs(sum) >= fabs(w)) comp += (sum - t) + w;
    else comp += (w - t) + sum;
    sum = t;
  }
  return (sum + comp) / (double)R;
}
double orc_adaptive_dbeta(int64_t R, const int32_t* E, double target, double dbeta_max, int iters) {
  if (orc_overlap(R, E, dbeta_max) >= target) return dbeta_max;
  double lo = 0.0, hi = dbeta_max; /* alpha(lo) >= target > alpha(hi) */
  for (int it = 0; it < iters; ++it) {
    double mid = 0.5 * (lo + hi);
    if (orc_overlap(R, E, mid) >= target) lo = mid;
    else hi = mid;
  }
  return lo;
}

/* ------------------------------------------------------------------------------------------
 * A5.  Offspring placement ("off-springs, as exact copies"; reading G5):
 * off_j = sum_{i<j} n_i, R' = off_R; child slots off_j .. off_j + n_j - 1 are copies of parent j.
 * ---------------------------------------------------------------------------------------- */
int64_t orc_exclusive_scan(int64_t R, const uint32_t* n, uint32_t* off /* R+1 */) {
  uint64_t run = 0;
  for (int64_t j = 0; j < R; ++j) {
    off[j] = (uint32_t)run;
    run += n[j];
  }
  off[R] = (uint32_t)run;
  return (int64_t)run; /* caller checks run < 2^32 and run <= capacity */
}

void orc_copy(int L, int64_t R, const uint32_t* n, const uint32_t* off, const uint32_t* src,
              const int32_t* Esrc, const int32_t* Msrc, uint32_t* dst, int32_t* Edst, int32_t* Mdst) {
  int64_t wpr = orc_words_per_replica(L);
#pragma omp parallel for schedule(dynamic, 1024)
  for (int64_t j = 0; j < R; ++j) {
    for (uint32_t c = 0; c < n[j]; ++c) {
      int64_t i = (int64_t)off[j] + c;
      for (int64_t w = 0; w < wpr; ++w) dst[i * wpr + w] = src[j * wpr + w];
      Edst[i] = Esrc[j];
      Mdst[i] = Msrc[j];
    }
  }
}

/* parent of every child by the plain definition: the unique j with off_j <= i < off_j + n_j */
void orc_parent_of(int64_t R, const uint32_t* n, const uint32_t* off, int64_t Rnew, uint32_t* parent) {
  for (int64_t j = 0; j < R; ++j)
    for (uint32_t c = 0; c < n[j]; ++c) parent[(int64_t)off[j] + c] = (uint32_t)j;
  (void)Rnew;
}

/* ------------------------------------------------------------------------------------------
 * A6.  Partition balancer: single-device analogue of the "main" algorithm.
 * Desired size r_p of partition p: counts differ by at most one replica;
 * born_p = offspring of the parents that lived in partition p (what a non-redistributing node
 * would hold); excess maxg_p = born_p - r_p or shortage minl_p = r_p - born_p,
 * "depending on case which one is positive".
 * ---------------------------------------------------------------------------------------- */
void orc_partition_table(int64_t Rpop, int P, uint32_t* part_start /* P+1 */) {
  int64_t base = Rpop / P, rem = Rpop % P;
  for (int p = 0; p <= P; ++p) part_start[p] = (uint32_t)(p * base + (p < rem ? p : rem));
}
/* stats[p*4 + {0,1,2,3}] = cnt_p, born_p, maxg_p, minl_p ; returns 'moved' */
int64_t orc_partition_stats(int64_t R, const uint32_t* n, const uint32_t* off, int P,
                            const uint32_t* old_start, const uint32_t* new_start, uint32_t* stats) {
  for (int p = 0; p < P; ++p) {
    uint32_t cnt = new_start[p + 1] - new_start[p];
    uint32_t born = off[old_start[p + 1]] - off[old_start[p]];
    stats[p * 4 + 0] = cnt;
    stats[p * 4 + 1] = born;
    stats[p * 4 + 2] = born > cnt ? born - cnt : 0u;
    stats[p * 4 + 3] = cnt > born ? cnt - born : 0u;
  }
  /* moved = children whose partition differs from their parent's partition */
  int64_t moved = 0;
  int pp = 0; /* partition of parent j: old_start[pp] <= j < old_start[pp+1] */
  int pc = 0; /* partition of child i (children are visited in increasing i) */
  for (int64_t j = 0; j < R; ++j) {
    while (pp + 1 < P && (int64_t)old_start[pp + 1] <= j) ++pp;
    for (uint32_t c = 0; c < n[j]; ++c) {
      int64_t i = (int64_t)off[j] + c;
      while (pc + 1 < P && (int64_t)new_start[pc + 1] <= i) ++pc;
      if (pc != pp) moved += 1;
    }
  }
  return moved;
}

/* ------------------------------------------------------------------------------------------
 * A6b.  Redistribution policies (readings G21-G23).  The children are in parent order;
 * partition p's parents produced born_p of them (a contiguous range); a policy chooses how many, cnt_p, each
 * partition holds afterwards (contiguous ranges again, sum cnt_p = R').
 *   policy 0  "balanced": r_p = floor(R'/P) + (p < R' mod P)  -- orc_partition_table above (counts differ <= 1 replica).
 *   policy 1  "main": replicas move in blocks of B; desired r_p as in policy 0; window W = maxexc * B.
 *             Start from cnt_p = born_p.  While some partition lies outside the window (cnt_p - r_p > W or
 *             r_p - cnt_p > W): move one block of B replicas from the partition with the largest excess cnt_p - r_p
 *             to the one with the largest shortage r_p - cnt_p (ties: lowest index).
 *   policy 2  "naive": every partition hands floor(born_p / 2) replicas -- a number proportional to its
 *             offspring -- to a common pool, and the pool is dealt back evenly: partition p receives
 *             floor(pool / P) + (p < pool mod P).
 *   policy 3  "none": cnt_p = born_p, nothing moves.
 * Returns the number of block moves made (policy 1), else 0.
 * ---------------------------------------------------------------------------------------- */
int64_t orc_policy_counts(int P, const uint32_t* born, int policy, uint32_t B, uint32_t maxexc, uint32_t* cnt) {
  int64_t Rnew = 0;
  for (int p = 0; p < P; ++p) Rnew += born[p];
  int64_t base = Rnew / P, rem = Rnew % P;
  if (policy == 0) {
    for (int p = 0; p < P; ++p) cnt[p] = (uint32_t)(base + (p < rem ? 1 : 0));
    return 0;
  }
  if (policy == 3) {
    for (int p = 0; p < P; ++p) cnt[p] = born[p];
    return 0;
  }
  if (policy == 2) {
    int64_t pool = 0;
    for (int p = 0; p < P; ++p) pool += born[p] / 2u;
    int64_t share = pool / P, extra = pool % P;
    for (int p = 0; p < P; ++p) cnt[p] = (uint32_t)((int64_t)born[p] - (int64_t)(born[p] / 2u) + share + (p < extra ? 1 : 0));
    return 0;
  }
  /* policy 1 */
  int64_t W = (int64_t)maxexc * (int64_t)B, moves = 0;
  int64_t* c = (int64_t*)malloc((size_t)P * sizeof(int64_t));
  for (int p = 0; p < P; ++p) c[p] = born[p];
  for (;;) {
    int hi = 0, lo = 0;
    int64_t e_hi = 0, e_lo = 0;
    for (int p = 0; p < P; ++p) {
      int64_t r = base + (p < rem ? 1 : 0);
      int64_t e = c[p] - r; /* excess (positive) or shortage (negative) */
      if (p == 0 || e > e_hi) { e_hi = e; hi = p; }
      if (p == 0 || e < e_lo) { e_lo = e; lo = p; }
    }
    if (e_hi <= W && -e_lo <= W) break; /* every partition inside the window */
    c[hi] -= (int64_t)B;
    c[lo] += (int64_t)B;
    moves += 1;
  }
  for (int p = 0; p < P; ++p) cnt[p] = (uint32_t)c[p];
  free(c);
  return moves;
}

/* partition table from counts: start[0] = 0, start[p+1] = start[p] + cnt[p] */
void orc_starts_from_counts(int P, const uint32_t* cnt, uint32_t* start /* P+1 */) {
  uint64_t run = 0;
  for (int p = 0; p < P; ++p) {
    start[p] = (uint32_t)run;
    run += cnt[p];
  }
  start[P] = (uint32_t)run;
}

/* ------------------------------------------------------------------------------------------
 * C4.  MCMC equilibration ("any traditional MCMC"; reading G7: checkerboard
 * Metropolis).  Thresholds T4/T8: floor(2^32 exp(-4 beta)), floor(2^32 exp(-8 beta)), clamped
 * to 2^32-1 (reading G10); accept iff dE <= 0 or u32 < T_dE (strict).
 * Random for an active site (C3, reading G20): ordinal q = y*(L/2) + k within the half-sweep,
 * x = 2k + ((y+colour)&1).  32 consecutive ordinals form a group gamma = q>>5, position p = q&31.  The group
 * owns 32 keyed words W_b, b = 0..31: W_b = word (b&3) of Philox counter (slot, 8*gamma + (b>>2), 2t+colour,
 * tag2|step).  The site's 32-bit uniform is the bit column p of those words, word 0 giving the most
 * significant bit:  u = sum_b bit_p(W_b) * 2^(31-b).
 * ---------------------------------------------------------------------------------------- */
void orc_thresholds(double beta, uint32_t* T4, uint32_t* T8) {
  double a4 = floor(4294967296.0 * exp(-4.0 * beta));
  double a8 = floor(4294967296.0 * exp(-8.0 * beta));
  *T4 = a4 >= 4294967295.0 ? 0xffffffffu : (uint32_t)a4;
  *T8 = a8 >= 4294967295.0 ? 0xffffffffu : (uint32_t)a8;
}

/* Jx, Jy: couplings of the +-J model (section D1 below), NULL = the ferromagnet of eq. (6) (every J = +1) */
static void sweeps_one_replica(int L, int8_t* s, uint64_t seed, uint32_t step, uint32_t slot, int theta,
                               uint32_t T4, uint32_t T8, const int8_t* Jx, const int8_t* Jy) {
  int half = L / 2;
  for (int t = 0; t < theta; ++t) {
    for (int colour = 0; colour < 2; ++colour) {
      uint32_t W[32]; /* the keyed words of the current group of 32 active sites */
      for (int y = 0; y < L; ++y) {
        for (int k = 0; k < half; ++k) {
          int x = 2 * k + ((y + colour) & 1);
          uint32_t q = (uint32_t)(y * half + k);
          uint32_t gamma = q >> 5, p = q & 31u;
          if (p == 0u) /* a new group starts: eight Philox blocks = 32 words */
            for (uint32_t c = 0; c < 8u; ++c)
              philox_keyed(seed, slot, 8u * gamma + c, (uint32_t)(2 * t + colour), TAG_SWEEP, step, W + 4 * c);
          uint32_t u = 0u; /* bit column p, W[0] most significant */
          for (int b = 0; b < 32; ++b) u |= ((W[b] >> p) & 1u) << (31 - b);
          int sig = s[y * L + x];
          int xr = (x + 1) % L, xl = (x + L - 1) % L, yd = (y + 1) % L, yu = (y + L - 1) % L;
          /* J_b * sigma_b of the four neighbours: right, left, down, up (the bond to the left neighbour is the
           * left neighbour's Jx, the bond to the upper neighbour is the upper neighbour's Jy) */
          int nb[4] = {s[y * L + xr], s[y * L + xl], s[yd * L + x], s[yu * L + x]};
          if (Jx) {
            nb[0] *= Jx[y * L + x];
            nb[1] *= Jx[y * L + xl];
            nb[2] *= Jy[y * L + x];
            nb[3] *= Jy[yu * L + x];
          }
          int a = 0; /* number of unsatisfied bonds of the site (anti-aligned neighbours when J = +1) */
          for (int d = 0; d < 4; ++d) a += (nb[d] != sig);
          int dE = 8 - 4 * a; /* = 2 sigma sum_b J_b sigma_b */
          int flip;
          if (dE <= 0) flip = 1;
          else if (dE == 4) flip = (u < T4);
          else flip = (u < T8);
          if (flip) s[y * L + x] = (int8_t)(-sig);
        }
      }
    }
  }
}

/* theta sweeps of replicas first..first+count-1 (slot index = position in the population) */
void orc_sweeps_J(int L, int64_t first, int64_t count, uint32_t* packed_base, uint64_t seed, uint32_t step,
                  int theta, uint32_t T4, uint32_t T8, const int8_t* Jx, const int8_t* Jy) {
  int64_t wpr = orc_words_per_replica(L);
#pragma omp parallel
  {
    int8_t* s = (int8_t*)malloc((size_t)L * L);
#pragma omp for schedule(static)
    for (int64_t i = first; i < first + count; ++i) {
      unpack_replica(L, packed_base + i * wpr, s);
      sweeps_one_replica(L, s, seed, step, (uint32_t)i, theta, T4, T8, Jx, Jy);
      pack_replica(L, s, packed_base + i * wpr);
    }
    free(s);
  }
}
void orc_sweeps(int L, int64_t first, int64_t count, uint32_t* packed_base, uint64_t seed, uint32_t step,
                int theta, uint32_t T4, uint32_t T8) {
  orc_sweeps_J(L, first, count, packed_base, seed, step, theta, T4, T8, NULL, NULL);
}

/* sweeps of an arbitrary list of slots, each given as its own packed lattice (used for the
 * sampled parity checks at full size: a replica's sweeps depend only on its lattice and slot) */
void orc_sweeps_slots_J(int L, int64_t count, const uint32_t* slots, uint32_t* packed_list, uint64_t seed,
                        uint32_t step, int theta, uint32_t T4, uint32_t T8, const int8_t* Jx, const int8_t* Jy) {
  int64_t wpr = orc_words_per_replica(L);
#pragma omp parallel
  {
    int8_t* s = (int8_t*)malloc((size_t)L * L);
#pragma omp for schedule(static)
    for (int64_t i = 0; i < count; ++i) {
      unpack_replica(L, packed_list + i * wpr, s);
      sweeps_one_replica(L, s, seed, step, slots[i], theta, T4, T8, Jx, Jy);
      pack_replica(L, s, packed_list + i * wpr);
    }
    free(s);
  }
}
void orc_sweeps_slots(int L, int64_t count, const uint32_t* slots, uint32_t* packed_list, uint64_t seed,
                      uint32_t step, int theta, uint32_t T4, uint32_t T8) {
  orc_sweeps_slots_J(L, count, slots, packed_list, seed, step, theta, T4, T8, NULL, NULL);
}

/* ------------------------------------------------------------------------------------------
 * A8.  Observables (reading G15): exact integer sums over the population of
 * E, E^2, |M|, M^2, M^4.  128-bit results as (lo, hi) pairs of uint64 (two's complement for sumE).
 * out[0..1]=sum E, [2..3]=sum E^2, [4..5]=sum |M|, [6..7]=sum M^2, [8..9]=sum M^4
 * ---------------------------------------------------------------------------------------- */
void orc_moment_sums(int64_t R, const int32_t* E, const int32_t* M, uint64_t* out) {
  __int128 sE = 0;
  unsigned __int128 sE2 = 0, sA = 0, sM2 = 0, sM4 = 0;
  for (int64_t j = 0; j < R; ++j) {
    int64_t e = E[j], m = M[j];
    uint64_t am = (uint64_t)(m < 0 ? -m : m);
    sE += e;
    sE2 += (unsigned __int128)((uint64_t)(e * e));
    sA += am;
    sM2 += (unsigned __int128)(am * am);
    sM4 += (unsigned __int128)(am * am) * (unsigned __int128)(am * am);
  }
  unsigned __int128 v[5] = {(unsigned __int128)sE, sE2, sA, sM2, sM4};
  for (int i = 0; i < 5; ++i) {
    out[2 * i] = (uint64_t)v[i];
    out[2 * i + 1] = (uint64_t)(v[i] >> 64);
  }
}

/* ------------------------------------------------------------------------------------------
 * Test helpers that are plain restatements (no method arithmetic beyond the above).
 * ---------------------------------------------------------------------------------------- */
/* energy of ONE replica given as int8 +-1 spins (for brute-force enumeration tests) */
int32_t orc_energy_int8(int L, const int8_t* s) { return energy_of(L, s); }
void orc_pack(int L, const int8_t* s, uint32_t* words) { pack_replica(L, s, words); }
void orc_unpack(int L, const uint32_t* words, int8_t* s) { unpack_replica(L, words, s); }
