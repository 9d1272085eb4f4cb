// pa_common.cuh -- device-side state, step parameters and the Philox4x32-10 generator.
// Part of the CUDA product path; shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace pa {

// ---------------------------------------------------------------------------------------------------
// Device-resident state of one context.  Every kernel of a step reads it; only single-thread epilogues
// write it.  A step is COMMITTED by k_observe's last block (cur ^= 1, R = Rnew, ...); when status != 0
// every later kernel returns at once, so a failed step leaves the population untouched.
// ---------------------------------------------------------------------------------------------------
struct DevState {
  unsigned long long R;          // current population R_beta_i
  unsigned long long Rnew;       // population after resampling (valid inside a step)
  unsigned long long R_parents;  // population the last committed step started from
  double sumw;                   // sum_j exp(-dbeta E_j)
  double Q;                      // eq. 3
  double lnQ;
  double sum_lnQ;                // eq. 5 accumulator
  double scale;                  // R0 / R  (reading G2)
  double beta;                   // inverse temperature of the current population
  unsigned long long moved;      // children whose partition differs from the parent's (last step)
  unsigned long long obs[10];    // {lo,hi} x (sum E, sum E^2, sum |M|, sum M^2, sum M^4)
  unsigned long long obs_R;
  unsigned long long replica_steps;  // sum over committed steps of R' (work counter for throughput metrics)
  unsigned int step;             // committed steps
  unsigned int cur;              // index of the buffer holding the current population
  unsigned int status;           // 0 = ok, else -pa_status of the failing step
  unsigned int fail_step;        // ordinal of the step that failed
  unsigned int reduce_done;      // block counters (reset every step by k_q_reduce)
  unsigned int scan_tile;        // ticket counter of k_poisson_scan
  unsigned int slot0;            // shard of a multi-GPU run: global index of local slot 0 of the CURRENT population (else 0)
  unsigned int slot0_new;        // ... of the population the running step builds
  unsigned int dist;             // 1: this context is one rank's shard (Q comes from all ranks; the step is committed in place)
  unsigned int pad2_[4];
  unsigned int scan_overflow;    // a parent sat on a level with lambda >= 2^31
  unsigned int obs_done;
  unsigned int T4, T8;           // thresholds of the last committed step with theta > 0
  int lev_lo, lev_hi;            // occupied energy levels (E + 2N)/4 of the CURRENT population, inclusive (by k_observe)
  int e_off;                     // E mod 4 of every configuration: 0 for the ferromagnet, 2 * (#negative bonds & 1) for a +-J sample
  double Q_committed;            // Q of the last COMMITTED step (Q above is overwritten by every attempt)
  double adaptive_dbeta;         // result of the last k_adaptive_step
};

struct StepParams {
  double dbeta;      // beta_next - beta (host fp64 subtraction, C5)
  double beta_next;
  unsigned int T4, T8;  // C4 thresholds at beta_next (host libm)
  int theta;
  int pad_;
};

// status codes stored in DevState::status (positive; the host negates them into pa_status)
enum { ST_OK = 0, ST_CAPACITY = 3, ST_EXTINCT = 4 };

// ---------------------------------------------------------------------------------------------------
// Philox4x32-10.  The key schedule depends only on the seed, so the ten round keys are computed once
// on the host and passed by value (they end up in the constant bank and feed LOP3 directly).
// ---------------------------------------------------------------------------------------------------
struct PhiloxKey {
  uint32_t k0[10];
  uint32_t k1[10];
};

constexpr uint32_t PHILOX_M0 = 0xD2511F53u;
constexpr uint32_t PHILOX_M1 = 0xCD9E8D57u;
constexpr uint32_t TAG_INIT = 0u, TAG_RESAMPLE = 1u, TAG_SWEEP = 2u;

__device__ __forceinline__ void philox_round(uint32_t& c0, uint32_t& c1, uint32_t& c2, uint32_t& c3, uint32_t k0,
                                             uint32_t k1) {
  const uint32_t hi0 = __umulhi(PHILOX_M0, c0), lo0 = PHILOX_M0 * c0;
  const uint32_t hi1 = __umulhi(PHILOX_M1, c2), lo1 = PHILOX_M1 * c2;
  const uint32_t n0 = hi1 ^ c1 ^ k0;
  const uint32_t n2 = hi0 ^ c3 ^ k1;
  c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
}

__device__ __forceinline__ uint4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                               const PhiloxKey& key) {
#pragma unroll
  for (int r = 0; r < 10; ++r) philox_round(c0, c1, c2, c3, key.k0[r], key.k1[r]);
  return make_uint4(c0, c1, c2, c3);
}

__device__ __forceinline__ uint32_t ctr3(uint32_t tag, uint32_t step) { return (tag << 28) | step; }

// E and M of a replica share ONE 32-bit word in HBM: floor(E / 4) in the upper half, M / 2 in the lower half.  Both are
// exact (E = e_off mod 4 with e_off = 0 for the ferromagnet, C1, and 0 or 2 for a +-J sample, D1; M = 2 popc - N
// with N even) and fit 16 bits for every supported lattice (|E / 4|, |M / 2| <= N / 2 = 8192 at L = 128).  Halves the E/M
// traffic of the reductions and of the redistribution copy; the energy level of C5 / A4 is simply the upper half + N / 2,
// and the energy of level lev is 4 lev - 2N + e_off.
__device__ __forceinline__ int32_t pack_em(int E, int M) {
  return (int32_t)(((uint32_t)(E >> 2) << 16) | ((uint32_t)(M >> 1) & 0xffffu));
}
__device__ __forceinline__ int em_energy(int32_t w, int e_off) { return (w >> 16) * 4 + e_off; }
__device__ __forceinline__ int em_level(int32_t w, int N) { return (w >> 16) + (N >> 1); }  // (E + 2N) / 4
__device__ __forceinline__ int em_mag(int32_t w) { return ((int32_t)((uint32_t)w << 16) >> 16) * 2; }

#ifndef PA_PDL_TRIGGER
#define PA_PDL_TRIGGER 0
#endif
#ifndef PA_PDL
#define PA_PDL 1
#endif
// Programmatic dependent launch: the kernels of a step are launched with programmatic stream serialisation, so a
// kernel's launch is staged while its predecessor runs; nothing the predecessor wrote is touched before this returns
// (a no-op when the kernel was launched without the attribute).  An early griddepcontrol.launch_dependents was
// measured SLOWER on B200 (config 5: a1-a6 0.738 ms with it, 0.679 ms without, 0.683 ms without PDL at all): the
// successor's blocks park on the SMs and take registers and warp slots from the kernel that still works.
__device__ __forceinline__ void grid_dependency_wait() {
#if PA_PDL_TRIGGER
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");  // the successor's blocks may be placed once all of ours have started
#endif
  asm volatile("griddepcontrol.wait;" ::: "memory");               // ... but nobody reads before the predecessor is complete
}

}  // namespace pa
