// pa_b200.cu -- C ABI of the population-annealing hot path (include/pa_b200.h) and its host-side step driver.
// Host logic only sequences kernels; every step a0-a8 of the path runs on the device.
#include "../../include/pa_b200.h"

#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <optional>
#include <string>
#include <algorithm>
#include <vector>

#include "pa_common.cuh"
#include "pa_observe.cuh"
#include "pa_resample.cuh"
#include "pa_sweep.cuh"

using namespace pa;

namespace {

constexpr int RUN_CHUNK = 1024;  // step-parameter slots uploaded per pa_run chunk
#ifndef PA_RED_GRID
#define PA_RED_GRID (148 * 4)
#endif
constexpr int RED_GRID = PA_RED_GRID;
constexpr int OBS_GRID = 148 * 4;

struct Layout {
  uint64_t state, params, spins[2], EM[2], off, n, tau, tile_desc, tile_parent, parent_of, red_partial, obs_partial,
      lev_tau, lev_mu, lev_m, lev_cdf, lev_hist, part[2], part_stats, bond_mask, ovl_hist, sys_tiles, dist_map, total;
};

inline uint64_t align_up(uint64_t x, uint64_t a) { return (x + a - 1) / a * a; }

int copy_tile_for(int L) {
  switch (L) {
    case 8: return CopyGeo<8>::CT;
    case 16: return CopyGeo<16>::CT;
    case 32: return CopyGeo<32>::CT;
    case 64: return CopyGeo<64>::CT;
    default: return CopyGeo<128>::CT;
  }
}

int copy_shift_for(int L) {  // CopyGeo<L>::CT is a power of two
  int sh = 0;
  while ((1 << sh) < copy_tile_for(L)) ++sh;
  return sh;
}

bool valid_L(int L) { return L == 8 || L == 16 || L == 32 || L == 64 || L == 128; }

int64_t default_capacity(int64_t R0) {
  int64_t s = (int64_t)std::ceil(std::sqrt((double)R0));
  while (s * s < R0) ++s;
  while (s > 0 && (s - 1) * (s - 1) >= R0) --s;
  int64_t slack = 16 * s;
  if (slack < 1024) slack = 1024;
  return (R0 + slack + 1023) / 1024 * 1024;
}

bool make_layout(const pa_config* c, int64_t cap, Layout* lo, bool shard = false) {
  if (!c || !valid_L(c->L) || c->P < 1 || c->R0 < 1 || c->R0 >= (1ll << 31) || cap < c->R0 || cap >= (1ll << 32) - 4096)
    return false;
  if (c->policy > PA_POLICY_NONE || (c->policy != PA_POLICY_BALANCED && c->P > BAL_PMAX)) return false;
  if ((c->flags & PA_RESAMPLE_NEAREST) && (c->flags & PA_RESAMPLE_SYSTEMATIC)) return false;  // one resampling rule
  const uint64_t N = (uint64_t)c->L * c->L, S = N / 8, nlev = N + 1, ucap = (uint64_t)cap;
  uint64_t o = 0;
  auto take = [&](uint64_t bytes) {
    const uint64_t at = o;
    o = align_up(o + bytes, 256);
    return at;
  };
  lo->state = take(sizeof(DevState));
  lo->params = take(sizeof(StepParams) * RUN_CHUNK);
  for (int b = 0; b < 2; ++b) lo->spins[b] = take(ucap * S + 64);  // + 64: the spare buffer doubles as the E / M staging area of pa_energies (8 n + 12 bytes at L = 8)
  for (int b = 0; b < 2; ++b) lo->EM[b] = take(ucap * 4);  // packed E/4 : M/2, one word per replica
  lo->off = take((ucap + 1) * 4);
  lo->n = (c->flags & (PA_KEEP_COUNTS | PA_RESAMPLE_SYSTEMATIC)) ? take(ucap * 4) : 0;  // A4c hands its counts to the scan through n
  lo->tau = (c->flags & PA_KEEP_TAU) ? take(ucap * 8) : 0;
  lo->tile_desc = take(((ucap + SCAN_TILE - 1) / SCAN_TILE + 1) * 8);
  lo->tile_parent = take((ucap / copy_tile_for(c->L) + 2) * 4);  // theta = 0: first parent of every copy tile
  lo->parent_of = take(ucap * 4);  // theta > 0: child -> parent map of the sweep's gather-on-load
  lo->red_partial = take(RED_GRID * 8);
  lo->obs_partial = take((uint64_t)OBS_GRID * 12 * 8);
  lo->lev_tau = take(nlev * 8);
  lo->lev_mu = take(nlev * 8);
  lo->lev_m = take(nlev * 4);
  lo->lev_cdf = take(nlev * PO_ROW * 8);
  lo->lev_hist = take(nlev * 4);  // level histogram of the adaptive temperature step (all zero between calls)
  for (int b = 0; b < 2; ++b) lo->part[b] = take(((uint64_t)c->P + 1) * 4);
  lo->part_stats = take((uint64_t)c->P * 16);
  lo->bond_mask = take(N / 2);        // +-J model: negative-bond masks, 2 colours x N/64 plane words x 4 bonds (pa_sweep.cuh)
  lo->ovl_hist = take(nlev * 8);      // overlap histogram (pa_overlap_hist)
  lo->sys_tiles = take(((ucap + SCAN_TILE - 1) / SCAN_TILE + 1) * 8);  // systematic resampling: tile sums / prefixes of Lam
  // a multi-GPU shard: the scan's child -> parent map of the rank's own offspring (parent_of then holds the map of the NEW
  // local population: own children + received lattices)
  lo->dist_map = shard ? take(ucap * 4) : 0;
  lo->total = o;
  return true;
}

struct EventPair {
  cudaEvent_t a, b;
  int kernel;
};

}  // namespace

struct pa_ctx {
  pa_config cfg;
  int64_t cap;
  int N, wrep, device;
  Layout lo;
  char* ws;
  cudaStream_t stream;
  PhiloxKey key;
  DevState* h_state;  // pinned mirror
  StepParams* h_params;  // pinned staging for uploads
  // host mirrors of committed state
  int64_t R, R_parents, steps;
  double beta, sum_lnQ, last_Q;
  int64_t launches;
  bool profile, profile_span;
  int nearest;  // resampling rule: 0 Poisson (A4), 1 PA_RESAMPLE_NEAREST (A4b), 2 PA_RESAMPLE_SYSTEMATIC (A4c)
  bool glass;   // pa_set_bonds: the +-J Hamiltonian (sweep kernels compiled with the coupling masks)
  int e_off;    // E mod 4 of every configuration (0 unless the sample has an odd number of negative bonds: 2)
  bool attempt_failed;  // the last pa_step / pa_run ended with an uncommitted step: off / n / tau hold that attempt
  // multi-GPU shard (pa_dist_*): rank = partition
  int rank, world;          // world = 0: not a shard
  int64_t g_R0;             // target population of the WHOLE run (= cfg.R0 unless this is a shard)
  int dist_phase;           // 0 idle, 1 after pa_dist_begin, 2 after pa_dist_resample
  int dist_theta;
  bool dist_lean;           // theta > 0: own children are gathered by the sweep's load, only crossing slices are packed
  int64_t dist_T;           // the rank's offspring of the step in flight
  int64_t dist_recv;        // lattices the rank receives (landed behind its parents in the current buffer)
  bool dist_packed;
  double dist_beta_next;
  bool dbg_thresholds;  // test hook: pa_debug_set_thresholds
  uint32_t dbg_T4, dbg_T8;
  int scan_grid_max[2];  // co-resident blocks of k_poisson_scan on this device: [0] theta = 0 variant, [1] map-writing variant
  unsigned red_grid, obs_grid;  // blocks of the two reductions: 4 per SM for large populations, fewer for small ones
  std::vector<EventPair> ev_used, ev_free;
  std::string err, launch_err;

  template <class T> T* dev(uint64_t off) const { return reinterpret_cast<T*>(ws + off); }
};

namespace {

int fail(pa_ctx* c, int code, const std::string& msg) {
  if (c) c->err = msg;
  return code;
}
int cuda_fail(pa_ctx* c, cudaError_t e, const char* what) {
  return fail(c, PA_ECUDA, std::string(what) + ": " + cudaGetErrorString(e));
}
#define CK(call)                                            \
  do {                                                      \
    cudaError_t e_ = (call);                                \
    if (e_ != cudaSuccess) return cuda_fail(c, e_, #call);  \
  } while (0)

struct Prof {  // records an event pair around one launch when profiling is on
  pa_ctx* c;
  EventPair ep;
  bool on;
  cudaStream_t s;
  // per-kernel pairs only with PA_PROFILE; the a1-a6 span pair (is_launch = false) also with PA_PROFILE_SPAN
  Prof(pa_ctx* c_, int kernel, bool is_launch = true)
      : c(c_), on(c_->profile || (!is_launch && c_->profile_span)), s(c_->stream) {
    if (is_launch) c->launches += 1;
    if (!on) return;
    if (!c->ev_free.empty()) {
      ep = c->ev_free.back();
      c->ev_free.pop_back();
    } else {
      if (cudaEventCreate(&ep.a) != cudaSuccess || cudaEventCreate(&ep.b) != cudaSuccess) {
        on = false;  // out of events: this launch goes unprofiled rather than recording into an invalid handle
        return;
      }
    }
    ep.kernel = kernel;
    cudaEventRecord(ep.a, s);
  }
  ~Prof() {
    if (!on) return;
    cudaEventRecord(ep.b, s);
    c->ev_used.push_back(ep);
  }
};

LevelTables tables(pa_ctx* c) {
  LevelTables t;
  t.tau = c->dev<double>(c->lo.lev_tau);
  t.mu = c->dev<double>(c->lo.lev_mu);
  t.m = c->dev<uint32_t>(c->lo.lev_m);
  t.cdf = c->dev<double>(c->lo.lev_cdf);
  return t;
}

SweepArgs sweep_args(int theta, uint32_t T4, uint32_t T8, int mode) {
  SweepArgs sa;
  for (int i = 0; i < 32; ++i) {  // threshold bits, most significant first, as LOP3 operands
    sa.a[i] = ((T4 >> (31 - i)) & 1u) ? 0xffffffffu : 0u;
    sa.b[i] = ((T8 >> (31 - i)) & 1u) ? 0xffffffffu : 0u;
  }
  for (int i = 0; i < 8; ++i) sa.kase[i] = 2u * ((T4 >> (31 - i)) & 1u) + ((T8 >> (31 - i)) & 1u);
  sa.theta = theta;
  sa.mode = mode;
  return sa;
}

// Every kernel of the path is launched with programmatic stream serialisation (PDL): its blocks may be placed while
// the predecessor drains and wait in griddepcontrol.wait (pa_common.cuh) until the predecessor's memory is visible.
template <class... KArgs, class... Args>
void launch(pa_ctx* c, const char* name, void (*kern)(KArgs...), unsigned grid, unsigned block, Args... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(grid);
  cfg.blockDim = dim3(block);
  cfg.dynamicSmemBytes = 0;
  cfg.stream = c->stream;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at;
  cfg.numAttrs = PA_PDL ? 1 : 0;
  const cudaError_t e = cudaLaunchKernelEx(&cfg, kern, KArgs(args)...);
  if (e != cudaSuccess && c->launch_err.empty())  // reported by the next sync_state
    c->launch_err = std::string(name) + ": " + cudaGetErrorString(e);
}

template <int L>
void launch_sweep_L(pa_ctx* c, const SweepArgs& sa) {
  uint32_t *s0 = c->dev<uint32_t>(c->lo.spins[0]), *s1 = c->dev<uint32_t>(c->lo.spins[1]);
  int32_t *em0 = c->dev<int32_t>(c->lo.EM[0]), *em1 = c->dev<int32_t>(c->lo.EM[1]);
  const DevState* st = c->dev<DevState>(c->lo.state);
  const uint32_t* parent_of = c->dev<uint32_t>(c->lo.parent_of);
  const uint4* bm = c->dev<uint4>(c->lo.bond_mask);
  if constexpr (L >= 64) {
    const unsigned grid = (unsigned)(((uint64_t)c->cap + Geo<L>::RPB - 1) / Geo<L>::RPB);
    if (c->glass) launch(c, "k_sweep", k_sweep<L, true>, grid, SWEEP_THREADS, st, s0, s1, em0, em1, c->key, sa, parent_of, bm);
    else launch(c, "k_sweep", k_sweep<L, false>, grid, SWEEP_THREADS, st, s0, s1, em0, em1, c->key, sa, parent_of, bm);
  } else {
    // a group of G lanes holds NR replicas: 8 when that still gives every SM its four blocks (one full wave), else 2
    constexpr int RPB8 = SWEEP_SMALL_THREADS / SGeo<L>::G * 8;  // replicas per block with NR = 8
    if ((uint64_t)c->cfg.R0 >= (uint64_t)RPB8 * 148 * 4) {
      const unsigned grid = (unsigned)(((uint64_t)c->cap + RPB8 - 1) / RPB8);
      if (c->glass) launch(c, "k_sweep_small", k_sweep_small<L, true, 8>, grid, SWEEP_SMALL_THREADS, st, s0, s1, em0, em1, c->key, sa, parent_of, bm);
      else launch(c, "k_sweep_small", k_sweep_small<L, false, 8>, grid, SWEEP_SMALL_THREADS, st, s0, s1, em0, em1, c->key, sa, parent_of, bm);
    } else {
      const uint64_t threads = ((uint64_t)c->cap + 1) / 2 * SGeo<L>::G;
      const unsigned grid = (unsigned)((threads + SWEEP_SMALL_THREADS - 1) / SWEEP_SMALL_THREADS);
      if (c->glass) launch(c, "k_sweep_small", k_sweep_small<L, true, 2>, grid, SWEEP_SMALL_THREADS, st, s0, s1, em0, em1, c->key, sa, parent_of, bm);
      else launch(c, "k_sweep_small", k_sweep_small<L, false, 2>, grid, SWEEP_SMALL_THREADS, st, s0, s1, em0, em1, c->key, sa, parent_of, bm);
    }
  }
}
// mode 2: theta sweeps of the resampled population (lattices gathered from the parents' slots); mode 1: energies only
void launch_sweep(pa_ctx* c, int theta, uint32_t T4, uint32_t T8, int mode) {
  Prof p(c, PA_K_SWEEP);
  const SweepArgs sa = sweep_args(theta, T4, T8, mode);
  switch (c->cfg.L) {
    case 8: launch_sweep_L<8>(c, sa); break;
    case 16: launch_sweep_L<16>(c, sa); break;
    case 32: launch_sweep_L<32>(c, sa); break;
    case 64: launch_sweep_L<64>(c, sa); break;
    default: launch_sweep_L<128>(c, sa); break;
  }
}

template <int L>
void launch_copy_L(pa_ctx* c) {
  const unsigned grid = (unsigned)((c->cap + CopyGeo<L>::CT - 1) / CopyGeo<L>::CT);
  launch(c, "k_copy", k_copy<L>, grid, COPY_THREADS, c->dev<DevState>(c->lo.state), c->dev<uint32_t>(c->lo.off),
         c->dev<uint32_t>(c->lo.tile_parent), c->dev<uint32_t>(c->lo.spins[0]), c->dev<uint32_t>(c->lo.spins[1]),
         c->dev<int32_t>(c->lo.EM[0]), c->dev<int32_t>(c->lo.EM[1]));
}
void launch_copy(pa_ctx* c) {
  Prof p(c, PA_K_COPY);
  switch (c->cfg.L) {
    case 8: launch_copy_L<8>(c); break;
    case 16: launch_copy_L<16>(c); break;
    case 32: launch_copy_L<32>(c); break;
    case 64: launch_copy_L<64>(c); break;
    default: launch_copy_L<128>(c); break;
  }
}

// mode 0: sums of the new population, a5 (partition table + diagnostics) and the commit of the step; mode 1: sums only
void launch_observe(pa_ctx* c, const StepParams* sp, int mode, bool shard_table = false) {
  Prof p(c, PA_K_OBSERVE);
  launch(c, "k_observe", k_observe, c->obs_grid, OBS_THREADS, c->dev<DevState>(c->lo.state), sp, c->dev<int32_t>(c->lo.EM[0]),
         c->dev<int32_t>(c->lo.EM[1]),
         c->dev<unsigned long long>(c->lo.obs_partial), mode, c->N, c->dev<uint32_t>(c->lo.off),
         c->dev<uint32_t>(c->lo.part[0]), c->dev<uint32_t>(c->lo.part[1]), c->dev<uint32_t>(c->lo.part_stats),
         // a shard keeps ONE local partition (cfg.policy acts between the ranks, on the host): its table is [0, R'] and
         // the offsets of the rank's own offspring do not add up to R', so the block-moving policies must not run on it
         shard_table ? BalanceArgs{1, PA_POLICY_BALANCED, 1024u, 1u}
                     : BalanceArgs{c->cfg.P, (int)c->cfg.policy, c->cfg.block ? c->cfg.block : 1024u, c->cfg.maxexc ? c->cfg.maxexc : 1u});
}

// persistent grid of k_poisson_scan: blocks per SM (occupancy of the variant) x SMs
unsigned scan_grid(pa_ctx* c, bool map) {
  int& g = c->scan_grid_max[map ? 1 : 0];
  if (g == 0) {
    int per_sm = 0, sms = 0;
    if (map) cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_poisson_scan<true, true, 0>, SCAN_THREADS, 0);
    else cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_poisson_scan<true, false, 0>, SCAN_THREADS, 0);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, c->device);
    g = (per_sm > 0 && sms > 0) ? per_sm * sms : 148 * 4;
  }
  const unsigned tiles_cap = (unsigned)((c->cap + SCAN_TILE - 1) / SCAN_TILE);
  return tiles_cap < (unsigned)g ? (tiles_cap ? tiles_cap : 1u) : (unsigned)g;
}

// k_poisson_scan<KEEP, MAP, RULE>: KEEP = parity getters want tau / n, MAP = the consumer is the sweep's gather-on-load
// (child -> parent map) rather than k_copy (first parent per copy tile), RULE = 0 Poisson, 1 nearest integers (A4b),
// 2 counts given by the systematic-resampling kernels (A4c)
template <bool KEEP, bool MAP>
void launch_scan_rule(pa_ctx* c, unsigned grid, DevState* st, const int32_t* E0, const int32_t* E1, const LevelTables& tb,
                      const ScanOut& out, int shift, unsigned long long cap) {
  if (c->nearest == 2) launch(c, "k_poisson_scan", k_poisson_scan<KEEP, MAP, 2>, grid, SCAN_THREADS, st, E0, E1, tb, c->N, out, shift, cap, c->key);
  else if (c->nearest == 1) launch(c, "k_poisson_scan", k_poisson_scan<KEEP, MAP, 1>, grid, SCAN_THREADS, st, E0, E1, tb, c->N, out, shift, cap, c->key);
  else launch(c, "k_poisson_scan", k_poisson_scan<KEEP, MAP, 0>, grid, SCAN_THREADS, st, E0, E1, tb, c->N, out, shift, cap, c->key);
}
void launch_scan(pa_ctx* c, bool keep, bool map, unsigned grid, DevState* st, const int32_t* E0, const int32_t* E1,
                 const LevelTables& tb, const ScanOut& out, int shift, unsigned long long cap) {
  if (keep && map) launch_scan_rule<true, true>(c, grid, st, E0, E1, tb, out, shift, cap);
  else if (keep) launch_scan_rule<true, false>(c, grid, st, E0, E1, tb, out, shift, cap);
  else if (map) launch_scan_rule<false, true>(c, grid, st, E0, E1, tb, out, shift, cap);
  else launch_scan_rule<false, false>(c, grid, st, E0, E1, tb, out, shift, cap);
}

// all kernels of one temperature step, parameters in device slot sp:
//   theta = 0:  k_q_reduce (+ level tables), k_poisson_scan, k_copy, k_observe (+ a5)
//   theta > 0:  k_q_reduce (+ level tables), k_poisson_scan (+ child -> parent map), k_sweep (gathers the lattices
//               itself), k_observe (+ a5)
void enqueue_step(pa_ctx* c, const StepParams* sp, const StepParams& hp) {
  const int theta = hp.theta;
  DevState* st = c->dev<DevState>(c->lo.state);
  const LevelTables tb = tables(c);
  const int N = c->N;
  const int n_desc = (int)((c->cap + SCAN_TILE - 1) / SCAN_TILE + 1);
  const int32_t *E0 = c->dev<int32_t>(c->lo.EM[0]), *E1 = c->dev<int32_t>(c->lo.EM[1]);
  std::optional<Prof> span;  // a1-a6 as one span on the stream (not a launch)
  span.emplace(c, PA_K_RESAMPLE_SPAN, false);
  {
    Prof p(c, PA_K_Q_REDUCE);  // also resets the step's counters and look-back descriptors
    launch(c, "k_q_reduce", k_q_reduce, c->red_grid, RED_THREADS, st, sp, E0, E1, N, c->dev<double>(c->lo.red_partial),
           (double)c->g_R0, c->dev<unsigned long long>(c->lo.tile_desc), n_desc, tb, c->nearest);
  }
  {
    // persistent blocks pull tiles from a ticket counter
    const bool keep = c->lo.n || c->lo.tau;
    ScanOut out;
    out.off = c->dev<uint32_t>(c->lo.off);
    out.n = c->lo.n ? c->dev<uint32_t>(c->lo.n) : nullptr;
    out.tau = c->lo.tau ? c->dev<double>(c->lo.tau) : nullptr;
    out.tile_desc = c->dev<unsigned long long>(c->lo.tile_desc);
    out.parent_of = c->dev<uint32_t>(c->lo.parent_of);
    out.tile_parent = c->dev<uint32_t>(c->lo.tile_parent);
    const int shift = copy_shift_for(c->cfg.L);
    const unsigned long long cap = (unsigned long long)c->cap;
    const unsigned grid = scan_grid(c, theta > 0);
    if (c->nearest == 2) {  // A4c: 64-bit prefix of Lam -> copy counts in out.n, which the scan then only places
      const unsigned ntiles = (unsigned)((c->cap + SCAN_TILE - 1) / SCAN_TILE);
      unsigned long long* tiles = c->dev<unsigned long long>(c->lo.sys_tiles);
      Prof p(c, PA_K_POISSON_SCAN);
      launch(c, "k_sys_tile_sums", k_sys_tile_sums, ntiles, SYS_THREADS, (const DevState*)st, E0, E1, tb, N, tiles);
      c->launches += 2;
      launch(c, "k_sys_scan_tiles", k_sys_scan_tiles, 1u, 1024u, (const DevState*)st, tiles, ntiles);
      launch(c, "k_sys_counts", k_sys_counts, ntiles, SYS_THREADS, (const DevState*)st, E0, E1, tb, N, (const unsigned long long*)tiles,
             out.n, c->key);
    }
    Prof p(c, PA_K_POISSON_SCAN);
    launch_scan(c, keep, theta > 0, grid, st, E0, E1, tb, out, shift, cap);
  }
  if (theta == 0) launch_copy(c);  // a6; with sweeps to follow it is fused into the sweep's load
  span.reset();
  if (theta > 0) launch_sweep(c, theta, hp.T4, hp.T8, 2);
  launch_observe(c, sp, 0);
}

__global__ void k_init_state(DevState* st, unsigned long long R, double beta0, uint32_t* part0, int P) {
  if (threadIdx.x == 0 && blockIdx.x == 0) {
    memset(st, 0, sizeof(DevState));
    st->R = R;
    st->R_parents = R;
    st->beta = beta0;
    st->Q = 1.0;
    st->Q_committed = 1.0;
  }
  const unsigned long long base = R / P, rem = R % P;
  for (int p = threadIdx.x; p <= P; p += blockDim.x)
    part0[p] = (uint32_t)((unsigned long long)p * base + ((unsigned long long)p < rem ? p : rem));
}
// test hook support: set R and rebuild the partition table of the current buffer
__global__ void k_set_population(DevState* st, unsigned long long R, uint32_t* part0, uint32_t* part1, int P) {
  if (threadIdx.x == 0) {
    st->R = R;
    st->obs_done = 0u;
  }
  uint32_t* part = st->cur ? part1 : part0;
  const unsigned long long base = R / P, rem = R % P;
  for (int p = threadIdx.x; p <= P; p += blockDim.x)
    part[p] = (uint32_t)((unsigned long long)p * base + ((unsigned long long)p < rem ? p : rem));
}
// multi-GPU shard: mark the context, set the global index of local slot 0
__global__ void k_dist_mark(DevState* st, unsigned slot0) {
  st->dist = 1u;
  st->slot0 = slot0;
  st->slot0_new = slot0;
}
// ... and the size / first global slot of the population the exchange has just delivered
__global__ void k_dist_set_new(DevState* st, unsigned long long count, unsigned slot0_new) {
  st->Rnew = count;
  st->slot0_new = slot0_new;
}
// Lean shard step (theta > 0).  The rank's T offspring are children j = 0..T-1 in child order with parents map[j].  Of
// these, [a, b) stay on the rank; [0, a) go to lower ranks and [b, T) to higher ranks: k_dist_pack gathers exactly those
// into the spare buffer in child order (= destination order), the send side of the exchange.
__global__ void __launch_bounds__(256)
k_dist_pack(const DevState* __restrict__ st, uint32_t* spins0, uint32_t* spins1, const uint32_t* __restrict__ map,
            const unsigned long long a, const unsigned long long b, const unsigned long long T, const int wrep) {
  const uint32_t* __restrict__ src = st->cur ? spins1 : spins0;
  uint32_t* __restrict__ dst = st->cur ? spins0 : spins1;
  const unsigned long long words = (a + (T - b)) * (unsigned long long)wrep;
  const unsigned long long stride = (unsigned long long)gridDim.x * blockDim.x;
  for (unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; i < words; i += stride) {
    const unsigned long long k = i / (unsigned)wrep, w = i % (unsigned)wrep;
    const unsigned long long j = k < a ? k : b + (k - a);
    dst[i] = src[(unsigned long long)map[j] * wrep + w];
  }
}
// ... and the gather map of the rank's NEW population for the sweep's load (mode 2), which reads the CURRENT buffer:
// slots [0, n_lo) came from lower ranks and were landed behind the R parents, slots [n_lo, n_lo + b - a) are the rank's own
// children (parents map[a ..]), the rest came from higher ranks.
__global__ void __launch_bounds__(256)
k_dist_compose(const uint32_t* __restrict__ map, uint32_t* __restrict__ parent_of, const unsigned long long n_new,
               const unsigned long long n_lo, const unsigned long long n_stay, const unsigned long long a,
               const unsigned long long R_old) {
  const unsigned long long stride = (unsigned long long)gridDim.x * blockDim.x;
  for (unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; i < n_new; i += stride) {
    uint32_t v;
    if (i < n_lo) v = (uint32_t)(R_old + i);
    else if (i < n_lo + n_stay) v = map[a + (i - n_lo)];
    else v = (uint32_t)(R_old + n_lo + (i - n_lo - n_stay));
    parent_of[i] = v;
  }
}
__global__ void k_set_e_off(DevState* st, int e_off) {
  st->e_off = e_off;
  st->obs_done = 0u;  // the population sums are taken again (k_observe's last-block counter)
}
__global__ void k_clear_status(DevState* st) {
  st->status = 0u;
  st->obs_done = 0u;
}

// a context is bound to the device that was current in pa_init
int bind_device(pa_ctx* c) {
  int dev = -1;
  if (cudaGetDevice(&dev) == cudaSuccess && dev == c->device) return PA_OK;
  CK(cudaSetDevice(c->device));
  return PA_OK;
}

// read the device state back (synchronises) and refresh the host mirrors
int sync_state(pa_ctx* c) {
  CK(cudaMemcpyAsync(c->h_state, c->dev<DevState>(c->lo.state), sizeof(DevState), cudaMemcpyDeviceToHost, c->stream));
  CK(cudaStreamSynchronize(c->stream));
  CK(cudaGetLastError());
  if (!c->launch_err.empty()) {
    const std::string msg = "kernel launch failed: " + c->launch_err;
    c->launch_err.clear();
    return fail(c, PA_ECUDA, msg);
  }
  const DevState& s = *c->h_state;
  c->R = (int64_t)s.R;
  c->R_parents = (int64_t)s.R_parents;
  c->steps = s.step;
  c->beta = s.beta;
  c->sum_lnQ = s.sum_lnQ;
  if (s.step > 0) c->last_Q = s.Q_committed;
  return PA_OK;
}

int status_to_code(pa_ctx* c) {
  const DevState& s = *c->h_state;
  if (s.status == ST_OK) return PA_OK;
  char buf[160];
  if (s.status == ST_CAPACITY) {
    snprintf(buf, sizeof buf, "step %u: resampled population R'=%llu exceeds capacity %lld (not committed)", s.fail_step,
             (unsigned long long)s.Rnew, (long long)c->cap);
    c->err = buf;
    return PA_ECAPACITY;
  }
  snprintf(buf, sizeof buf, "step %u: population extinct (R'=0, not committed)", s.fail_step);
  c->err = buf;
  return PA_EEXTINCT;
}

int copy_out(pa_ctx* c, void* dst, const void* src_dev, size_t bytes, int dst_on_device) {
  if (bytes == 0) return PA_OK;
  if (int rc = bind_device(c)) return rc;
  CK(cudaMemcpyAsync(dst, src_dev, bytes, dst_on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, c->stream));
  CK(cudaStreamSynchronize(c->stream));
  return PA_OK;
}

int check_step_args(pa_ctx* c, double beta_from, double beta_next, int theta) {
  if (!(beta_next == beta_next) || std::isinf(beta_next)) return fail(c, PA_EINVAL, "beta_next is not finite");
  if (theta < 0) return fail(c, PA_EINVAL, "theta < 0");
  if (theta > 0 && beta_next < 0.0) return fail(c, PA_EINVAL, "beta_next < 0 with theta > 0 (reading G10)");
  const double dbeta = beta_next - beta_from;
  if (!(std::fabs(dbeta) * 2.0 * c->N < 700.0)) return fail(c, PA_EINVAL, "|dbeta|*2N >= 700 (reading G11)");
  return PA_OK;
}

StepParams make_params(const pa_ctx* c, double beta_from, double beta_next, int theta) {
  StepParams p;
  p.dbeta = beta_next - beta_from;
  p.beta_next = beta_next;
  const double a4 = std::floor(4294967296.0 * std::exp(-4.0 * beta_next));
  const double a8 = std::floor(4294967296.0 * std::exp(-8.0 * beta_next));
  p.T4 = a4 >= 4294967295.0 ? 0xffffffffu : (a4 > 0.0 ? (uint32_t)a4 : 0u);
  p.T8 = a8 >= 4294967295.0 ? 0xffffffffu : (a8 > 0.0 ? (uint32_t)a8 : 0u);
  if (c->dbg_thresholds) {
    p.T4 = c->dbg_T4;
    p.T8 = c->dbg_T8;
  }
  p.theta = theta;
  p.pad_ = 0;
  return p;
}

}  // namespace

extern "C" {

uint64_t pa_workspace_bytes(const pa_config* cfg) {
  if (!cfg) return 0;
  const int64_t cap = cfg->capacity > 0 ? cfg->capacity : (cfg->R0 >= 1 ? default_capacity(cfg->R0) : 0);
  Layout lo;
  if (!make_layout(cfg, cap, &lo)) return 0;
  return lo.total;
}

namespace {
// shared by pa_init (world = 0) and pa_dist_init (world >= 1: cfg holds the rank's local R0, global values in g_*)
int init_common(const pa_config* cfg, pa_ctx** out, int rank, int world, int64_t g_R0, int64_t g_first) {
  if (!cfg || !out) return PA_EINVAL;
  *out = nullptr;
  pa_ctx* c = new (std::nothrow) pa_ctx();
  if (!c) return PA_ENOMEM;
  c->cfg = *cfg;
  c->cap = cfg->capacity > 0 ? cfg->capacity : (cfg->R0 >= 1 ? default_capacity(cfg->R0) : 0);
  if (!make_layout(cfg, c->cap, &c->lo, world > 0) || !(cfg->beta0 == cfg->beta0)) {
    delete c;
    return PA_EINVAL;
  }
  if (!cfg->workspace || cfg->workspace_bytes < c->lo.total || ((uintptr_t)cfg->workspace & 255u)) {
    delete c;
    return cfg->workspace && !((uintptr_t)cfg->workspace & 255u) ? PA_ENOMEM : PA_EINVAL;
  }
  c->N = cfg->L * cfg->L;
  c->wrep = c->N / 32;
  c->ws = static_cast<char*>(cfg->workspace);
  c->stream = static_cast<cudaStream_t>(cfg->stream);
  c->profile = (cfg->flags & PA_PROFILE) != 0;
  c->profile_span = (cfg->flags & PA_PROFILE_SPAN) != 0;
  c->nearest = (cfg->flags & PA_RESAMPLE_SYSTEMATIC) ? 2 : ((cfg->flags & PA_RESAMPLE_NEAREST) ? 1 : 0);
  c->glass = false;
  c->e_off = 0;
  c->launches = 0;
  {  // a small population (config 1: 1024 replicas) is latency-bound: one block per 4096 replicas, at most 4 per SM
    const int64_t want = (c->cap + 4095) / 4096;
    c->red_grid = (unsigned)(want < 1 ? 1 : (want > RED_GRID ? RED_GRID : want));
    c->obs_grid = (unsigned)(want < 1 ? 1 : (want > OBS_GRID ? OBS_GRID : want));
  }
  c->attempt_failed = false;
  c->rank = 0;
  c->world = 0;
  c->dist_phase = 0;
  c->dist_lean = false;
  c->dist_packed = false;
  c->dist_T = 0;
  c->dist_recv = 0;
  c->dbg_thresholds = false;
  c->dbg_T4 = c->dbg_T8 = 0u;
  c->scan_grid_max[0] = c->scan_grid_max[1] = 0;
  uint32_t k0 = (uint32_t)(cfg->seed & 0xffffffffull), k1 = (uint32_t)(cfg->seed >> 32);
  for (int r = 0; r < 10; ++r) {
    c->key.k0[r] = k0;
    c->key.k1[r] = k1;
    k0 += 0x9E3779B9u;
    k1 += 0xBB67AE85u;
  }
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
    delete c;
    return PA_ECUDA;  // no CPU fallback
  }
  cudaGetDevice(&c->device);
  c->h_state = nullptr;
  c->h_params = nullptr;
  if (cudaHostAlloc((void**)&c->h_state, sizeof(DevState), cudaHostAllocDefault) != cudaSuccess ||
      cudaHostAlloc((void**)&c->h_params, sizeof(StepParams) * RUN_CHUNK, cudaHostAllocDefault) != cudaSuccess) {
    if (c->h_state) cudaFreeHost(c->h_state);
    delete c;
    return PA_ECUDA;
  }
  *out = c;  // from here on errors keep the ctx so that pa_last_error works; caller destroys it
  DevState* st = c->dev<DevState>(c->lo.state);
  k_init_state<<<1, 256, 0, c->stream>>>(st, (unsigned long long)cfg->R0, cfg->beta0, c->dev<uint32_t>(c->lo.part[0]),
                                         cfg->P);
  c->launches += 1;
  c->rank = rank;
  c->world = world;
  c->g_R0 = world > 0 ? g_R0 : cfg->R0;
  if (world > 0) {
    k_dist_mark<<<1, 1, 0, c->stream>>>(st, (unsigned)g_first);
    c->launches += 1;
  }
  CK(cudaMemsetAsync(c->dev<char>(c->lo.part_stats), 0, (size_t)cfg->P * 16, c->stream));
  CK(cudaMemsetAsync(c->dev<char>(c->lo.lev_hist), 0, ((size_t)c->N + 1) * 4, c->stream));
  {
    const int bpr = (c->wrep + 3) / 4;
    const uint64_t threads = (uint64_t)cfg->R0 * bpr;
    k_init<<<(unsigned)((threads + 255) / 256), 256, 0, c->stream>>>(st, c->dev<uint32_t>(c->lo.spins[0]),
                                                                      c->dev<uint32_t>(c->lo.spins[1]), c->wrep, c->key);
    c->launches += 1;
  }
  launch_sweep(c, 0, 0u, 0u, 1);   // E_j, M_j
  launch_observe(c, nullptr, 1);  // population sums
  c->last_Q = 1.0;
  int rc = sync_state(c);
  if (rc != PA_OK) return rc;
  return PA_OK;
}
}  // namespace

int pa_init(const pa_config* cfg, pa_ctx** out) { return init_common(cfg, out, 0, 0, 0, 0); }

int pa_run(pa_ctx* c, const double* betas, int32_t K, int32_t theta, int32_t* steps_done) {
  if (!c) return PA_EINVAL;
  if (steps_done) *steps_done = 0;
  if (K < 0 || (K > 0 && !betas)) return fail(c, PA_EINVAL, "bad betas/K");
  if (c->world > 0) return fail(c, PA_EINVAL, "this context is a multi-GPU shard: step it with pa_dist_begin / _resample / _finish");
  if (int rc = bind_device(c)) return rc;
  double from = c->beta;
  for (int k = 0; k < K; ++k) {
    const int rc = check_step_args(c, from, betas[k], theta);
    if (rc != PA_OK) return rc;
    from = betas[k];
  }
  if ((uint64_t)c->steps + (uint64_t)K >= (1ull << 28)) return fail(c, PA_EINVAL, "step counter would exceed 2^28");
  const int64_t steps_before = c->steps;
  StepParams* d_params = c->dev<StepParams>(c->lo.params);
  from = c->beta;
  for (int base = 0; base < K; base += RUN_CHUNK) {
    const int nk = (K - base < RUN_CHUNK) ? (K - base) : RUN_CHUNK;
    if (base > 0) CK(cudaStreamSynchronize(c->stream));  // staging buffer is reused
    for (int k = 0; k < nk; ++k) {
      c->h_params[k] = make_params(c, from, betas[base + k], theta);
      from = betas[base + k];
    }
    CK(cudaMemcpyAsync(d_params, c->h_params, sizeof(StepParams) * nk, cudaMemcpyHostToDevice, c->stream));
    for (int k = 0; k < nk; ++k) enqueue_step(c, d_params + k, c->h_params[k]);
  }
  int rc = sync_state(c);
  if (rc != PA_OK) return rc;
  if (steps_done) *steps_done = (int32_t)(c->steps - steps_before);
  rc = status_to_code(c);
  c->attempt_failed = (rc != PA_OK);
  if (rc != PA_OK) {
    k_clear_status<<<1, 1, 0, c->stream>>>(c->dev<DevState>(c->lo.state));
    c->launches += 1;
    CK(cudaStreamSynchronize(c->stream));
  }
  return rc;
}

int pa_step(pa_ctx* c, double beta_next, int32_t theta) { return pa_run(c, &beta_next, 1, theta, nullptr); }

int pa_population(pa_ctx* c, int64_t* R) {
  if (!c || !R) return PA_EINVAL;
  *R = c->R;
  return PA_OK;
}

int pa_totals(pa_ctx* c, int64_t* replica_steps) {
  if (!c || !replica_steps) return PA_EINVAL;
  *replica_steps = (int64_t)c->h_state->replica_steps;
  return PA_OK;
}

int pa_beta(pa_ctx* c, double* beta, int64_t* steps) {
  if (!c) return PA_EINVAL;
  if (beta) *beta = c->beta;
  if (steps) *steps = c->steps;
  return PA_OK;
}

int pa_energies(pa_ctx* c, int32_t* E, int32_t* M, int64_t n, int dst_on_device) {
  if (!c || n < 0 || n > c->R || (!E && !M)) return fail(c, PA_EINVAL, "pa_energies: bad arguments");
  if (n == 0) return PA_OK;
  if (c->dist_phase != 0) return fail(c, PA_EINVAL, "pa_energies: a multi-GPU step is in flight (the spare buffer is in use)");
  if (int rc = bind_device(c)) return rc;
  const unsigned cur = c->h_state->cur;
  const int32_t* em = c->dev<int32_t>(c->lo.EM[cur]);
  const unsigned grid = (unsigned)((n + 255) / 256);
  if (dst_on_device) {
    k_unpack_em<<<grid, 256, 0, c->stream>>>(em, E, M, (unsigned long long)n, c->e_off);
    c->launches += 1;
    CK(cudaStreamSynchronize(c->stream));
    return PA_OK;
  }
  // host destination: unpack into the spare population buffer (free outside a step; cap * S >= 8 n bytes), then copy
  int32_t* sE = c->dev<int32_t>(c->lo.spins[cur ^ 1u]);
  int32_t* sM = sE + ((n + 3) / 4) * 4;
  k_unpack_em<<<grid, 256, 0, c->stream>>>(em, E ? sE : nullptr, M ? sM : nullptr, (unsigned long long)n, c->e_off);
  c->launches += 1;
  int rc = PA_OK;
  if (E) rc = copy_out(c, E, sE, (size_t)n * 4, 0);
  if (rc == PA_OK && M) rc = copy_out(c, M, sM, (size_t)n * 4, 0);
  return rc;
}

int pa_log_Z(pa_ctx* c, double* lnZ, double* sum_lnQ, double* last_Q) {
  if (!c) return PA_EINVAL;
  if (lnZ) *lnZ = (double)c->N * std::log(2.0) + c->sum_lnQ;
  if (sum_lnQ) *sum_lnQ = c->sum_lnQ;
  if (last_Q) *last_Q = c->last_Q;
  return PA_OK;
}

int pa_observables(pa_ctx* c, pa_obs* o) {
  if (!c || !o) return PA_EINVAL;
  const DevState& s = *c->h_state;
  o->R = (int64_t)s.obs_R;
  o->sum_E = (int64_t)s.obs[0];
  for (int i = 0; i < 2; ++i) {
    o->sum_E2[i] = s.obs[2 + i];
    o->sum_absM[i] = s.obs[4 + i];
    o->sum_M2[i] = s.obs[6 + i];
    o->sum_M4[i] = s.obs[8 + i];
  }
  const double R = (double)s.obs_R;
  auto f = [](const unsigned long long* p) { return (double)p[0] + 18446744073709551616.0 * (double)p[1]; };
  o->mean_E = (double)o->sum_E / R;
  o->mean_E2 = f(&s.obs[2]) / R;
  o->mean_absM = f(&s.obs[4]) / R;
  o->mean_M2 = f(&s.obs[6]) / R;
  o->mean_M4 = f(&s.obs[8]) / R;
  return PA_OK;
}

int pa_spins(pa_ctx* c, uint32_t* dst, int64_t first, int64_t count, int dst_on_device) {
  if (!c || !dst || first < 0 || count < 0 || first + count > c->R) return fail(c, PA_EINVAL, "pa_spins: bad range");
  const unsigned cur = c->h_state->cur;
  return copy_out(c, dst, c->dev<uint32_t>(c->lo.spins[cur]) + (size_t)first * c->wrep, (size_t)count * c->wrep * 4,
                  dst_on_device);
}

int pa_tau(pa_ctx* c, double* dst, int64_t n, int dst_on_device) {
  if (!c || !dst || n < 0) return fail(c, PA_EINVAL, "pa_tau: bad arguments");
  if (!c->lo.tau) return fail(c, PA_EINVAL, "pa_tau needs PA_KEEP_TAU");
  if (c->steps == 0 || n > c->R_parents) return fail(c, PA_EINVAL, "pa_tau: no step yet or n > parents");
  if (c->attempt_failed) return fail(c, PA_EINVAL, "pa_tau: the last step was not committed (its tau array is not that of the last committed step)");
  return copy_out(c, dst, c->dev<double>(c->lo.tau), (size_t)n * 8, dst_on_device);
}

int pa_counts(pa_ctx* c, uint32_t* n, uint32_t* off, int64_t n_parents, int dst_on_device) {
  if (!c || n_parents < 0 || (!n && !off)) return fail(c, PA_EINVAL, "pa_counts: bad arguments");
  if (c->steps == 0 || n_parents > c->R_parents) return fail(c, PA_EINVAL, "pa_counts: no step yet or n_parents > parents");
  if (n && !c->lo.n) return fail(c, PA_EINVAL, "pa_counts(n) needs PA_KEEP_COUNTS");
  if (c->attempt_failed) return fail(c, PA_EINVAL, "pa_counts: the last step was not committed (off / n hold the failed attempt)");
  int rc = PA_OK;
  if (n) rc = copy_out(c, n, c->dev<uint32_t>(c->lo.n), (size_t)n_parents * 4, dst_on_device);
  if (rc == PA_OK && off) rc = copy_out(c, off, c->dev<uint32_t>(c->lo.off), (size_t)(n_parents + 1) * 4, dst_on_device);
  return rc;
}

int pa_parents(pa_ctx* c, int64_t* n_parents) {
  if (!c || !n_parents) return PA_EINVAL;
  *n_parents = c->R_parents;
  return PA_OK;
}

int pa_partitions(pa_ctx* c, uint32_t* part_start, pa_part_stats* stats, int64_t* moved) {
  if (!c || !part_start) return fail(c, PA_EINVAL, "pa_partitions: bad arguments");
  const unsigned cur = c->h_state->cur;
  int rc = copy_out(c, part_start, c->dev<uint32_t>(c->lo.part[cur]), ((size_t)c->cfg.P + 1) * 4, 0);
  if (rc == PA_OK && stats) rc = copy_out(c, stats, c->dev<uint32_t>(c->lo.part_stats), (size_t)c->cfg.P * 16, 0);
  if (moved) *moved = (int64_t)c->h_state->moved;
  return rc;
}

int pa_thresholds(pa_ctx* c, uint32_t* T4, uint32_t* T8) {
  if (!c) return PA_EINVAL;
  if (T4) *T4 = c->h_state->T4;
  if (T8) *T8 = c->h_state->T8;
  return PA_OK;
}

int pa_adaptive_beta(pa_ctx* c, double target_overlap, double dbeta_max, double* beta_next) {
  if (!c || !beta_next) return PA_EINVAL;
  if (!(target_overlap > 0.0 && target_overlap < 1.0) || !(dbeta_max > 0.0) || !(dbeta_max * 2.0 * c->N < 700.0))
    return fail(c, PA_EINVAL, "pa_adaptive_beta: need 0 < target < 1 and 0 < dbeta_max with dbeta_max*2N < 700");
  if (c->world > 0) return fail(c, PA_EINVAL, "pa_adaptive_beta: not available on a multi-GPU shard");
  if (int rc = bind_device(c)) return rc;
  DevState* st = c->dev<DevState>(c->lo.state);
  unsigned* hist = c->dev<unsigned>(c->lo.lev_hist);
  k_level_hist<<<c->obs_grid, OBS_THREADS, 0, c->stream>>>(st, c->dev<int32_t>(c->lo.EM[0]), c->dev<int32_t>(c->lo.EM[1]), hist, c->N);
  k_adaptive_step<<<1, OBS_THREADS, 0, c->stream>>>(st, hist, c->N, target_overlap, dbeta_max, 40);
  c->launches += 2;
  if (int rc = sync_state(c)) return rc;
  *beta_next = c->beta + c->h_state->adaptive_dbeta;
  return PA_OK;
}

int pa_debug_set_thresholds(pa_ctx* c, int enable, uint32_t T4, uint32_t T8) {
  if (!c) return PA_EINVAL;
  c->dbg_thresholds = enable != 0;
  c->dbg_T4 = T4;
  c->dbg_T8 = T8;
  return PA_OK;
}

int pa_set_spins(pa_ctx* c, const uint32_t* src, int64_t R, int src_on_device) {
  if (!c || !src || R < 1 || R > c->cap) return fail(c, PA_EINVAL, "pa_set_spins: bad arguments");
  if (int rc = bind_device(c)) return rc;
  const unsigned cur = c->h_state->cur;
  CK(cudaMemcpyAsync(c->dev<uint32_t>(c->lo.spins[cur]), src, (size_t)R * c->wrep * 4,
                     src_on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, c->stream));
  k_set_population<<<1, 256, 0, c->stream>>>(c->dev<DevState>(c->lo.state), (unsigned long long)R,
                                             c->dev<uint32_t>(c->lo.part[0]), c->dev<uint32_t>(c->lo.part[1]), c->cfg.P);
  c->launches += 1;
  launch_sweep(c, 0, 0u, 0u, 1);
  launch_observe(c, nullptr, 1);
  return sync_state(c);
}

// ---- second Hamiltonian: the 2D +-J spin glass (D1) -----------------------------
int pa_set_bonds(pa_ctx* c, const uint32_t* Jx, const uint32_t* Jy) {
  if (!c || ((Jx == nullptr) != (Jy == nullptr))) return fail(c, PA_EINVAL, "pa_set_bonds: give both coupling planes or neither");
  if (c->steps != 0 || c->dist_phase != 0) return fail(c, PA_EINVAL, "pa_set_bonds: only before the first temperature step");
  if (int rc = bind_device(c)) return rc;
  const int L = c->cfg.L, N = c->N, HB = L / 2, groups = N / 64;
  int e_off = 0;
  if (Jx) {
    // coupling of the bond that leaves site (x, y) to the right (Jx) / downwards (Jy): bit 1 <-> J = +1
    auto neg = [&](const uint32_t* J, int x, int y) {
      const int b = ((y + L) % L) * L + ((x + L) % L);
      return ((J[b >> 5] >> (b & 31)) & 1u) == 0u;
    };
    std::vector<uint32_t> mask((size_t)2 * groups * 4, 0u);
    int nneg = 0;
    for (int b = 0; b < N; ++b) nneg += (int)neg(Jx, b % L, b / L) + (int)neg(Jy, b % L, b / L);
    e_off = 2 * (nneg & 1);
    for (int C = 0; C < 2; ++C)
      for (int y = 0; y < L; ++y)
        for (int k = 0; k < HB; ++k) {
          const int odd = (y + C) & 1, x = 2 * k + odd;     // the active site (pa_sweep.cuh: plane C of row y, bit k)
          const int q = y * HB + k;                         // its ordinal in the half-sweep: group q >> 5, bit q & 31
          uint32_t* m = &mask[((size_t)C * groups + (q >> 5)) * 4];
          const uint32_t bit = 1u << (q & 31);
          if (neg(Jy, x, y - 1)) m[0] |= bit;               // up: the bond below (x, y-1)
          if (neg(Jy, x, y)) m[1] |= bit;                   // down
          // same plane bit k of the other colour is x+1 on an even (y+C), x-1 on an odd one; the shifted bit is the other side
          if (neg(Jx, odd ? x - 1 : x, y)) m[2] |= bit;
          if (neg(Jx, odd ? x : x - 1, y)) m[3] |= bit;
        }
    CK(cudaMemcpyAsync(c->dev<char>(c->lo.bond_mask), mask.data(), mask.size() * 4, cudaMemcpyHostToDevice, c->stream));
    CK(cudaStreamSynchronize(c->stream));  // `mask` is pageable host memory that dies with this scope
  }
  c->glass = Jx != nullptr;
  c->e_off = e_off;
  k_set_e_off<<<1, 1, 0, c->stream>>>(c->dev<DevState>(c->lo.state), e_off);
  c->launches += 1;
  launch_sweep(c, 0, 0u, 0u, 1);   // E_j, M_j of the current population under the new Hamiltonian
  launch_observe(c, nullptr, 1);
  return sync_state(c);
}

int pa_overlap_hist(pa_ctx* c, uint64_t* hist) {
  if (!c || !hist) return fail(c, PA_EINVAL, "pa_overlap_hist: bad arguments");
  if (c->world > 0) return fail(c, PA_EINVAL, "pa_overlap_hist: not available on a multi-GPU shard (partners live on other ranks)");
  if (int rc = bind_device(c)) return rc;
  unsigned long long* d_hist = c->dev<unsigned long long>(c->lo.ovl_hist);
  CK(cudaMemsetAsync(d_hist, 0, ((size_t)c->N + 1) * 8, c->stream));
  const int64_t pairs = c->R / 2;
  int64_t want = (pairs + 63) / 64;  // 8 pairs per block pass
  const unsigned grid = (unsigned)(want < 1 ? 1 : (want > 148 * 8 ? 148 * 8 : want));
  k_overlap_hist<<<grid, OVL_THREADS, 0, c->stream>>>(c->dev<DevState>(c->lo.state), c->dev<uint32_t>(c->lo.spins[0]),
                                                     c->dev<uint32_t>(c->lo.spins[1]), d_hist, c->N);
  c->launches += 1;
  return copy_out(c, hist, d_hist, ((size_t)c->N + 1) * 8, 0);
}

// ---- multi-GPU: partitioned redistribution ------------------------------------------------------------
namespace {
// balanced table value: start of partition p of `total` items over P partitions
inline int64_t balanced_start(int64_t total, int P, int p) {
  const int64_t base = total / P, rem = total % P;
  return (int64_t)p * base + (p < rem ? p : rem);
}
// counts under a policy from the per-rank offspring totals (host mirror of balance_tile; A6b)
void policy_counts_host(int P, const int64_t* born, int policy, uint32_t B, uint32_t maxexc, std::vector<int64_t>& cnt) {
  int64_t total = 0;
  for (int p = 0; p < P; ++p) total += born[p];
  const int64_t base = total / P, rem = total % P;
  cnt.assign(P, 0);
  if (policy == PA_POLICY_NONE) {
    for (int p = 0; p < P; ++p) cnt[p] = born[p];
  } else if (policy == PA_POLICY_NAIVE) {
    int64_t pool = 0;
    for (int p = 0; p < P; ++p) pool += born[p] / 2;
    const int64_t share = pool / P, extra = pool % P;
    for (int p = 0; p < P; ++p) cnt[p] = born[p] - born[p] / 2 + share + (p < extra ? 1 : 0);
  } else if (policy == PA_POLICY_MAIN) {
    const int64_t W = (int64_t)maxexc * (int64_t)B;
    for (int p = 0; p < P; ++p) cnt[p] = born[p];
    for (;;) {
      int hi = 0, lo = 0;
      int64_t e_hi = 0, e_lo = 0;
      for (int p = 0; p < P; ++p) {
        const int64_t e = cnt[p] - (base + (p < rem ? 1 : 0));
        if (p == 0 || e > e_hi) { e_hi = e; hi = p; }
        if (p == 0 || e < e_lo) { e_lo = e; lo = p; }
      }
      if (e_hi <= W && -e_lo <= W) break;
      cnt[hi] -= (int64_t)B;
      cnt[lo] += (int64_t)B;
    }
  } else {
    for (int p = 0; p < P; ++p) cnt[p] = base + (p < rem ? 1 : 0);
  }
}
}  // namespace

int pa_dist_exchange_plan(int32_t world, const int64_t* T, int32_t policy, uint32_t block, uint32_t maxexc,
                          int64_t* new_start, int64_t* base, int64_t* counts) {
  if (world < 1 || !T || !new_start || !base || !counts || policy < 0 || policy > PA_POLICY_NONE) return PA_EINVAL;
  for (int r = 0; r < world; ++r)
    if (T[r] < 0) return PA_ECAPACITY;
  std::vector<int64_t> cnt;
  policy_counts_host(world, T, policy, block ? block : 1024u, maxexc ? maxexc : 1u, cnt);
  base[0] = 0;
  new_start[0] = 0;
  for (int r = 0; r < world; ++r) {
    base[r + 1] = base[r] + T[r];
    new_start[r + 1] = new_start[r] + cnt[r];
  }
  if (base[world] == 0) return PA_EEXTINCT;
  // rank src's offspring are the global children [base[src], base[src+1]); rank dst's new range is
  // [new_start[dst], new_start[dst+1]): the slice is the intersection (contiguous on both sides)
  for (int src = 0; src < world; ++src)
    for (int dst = 0; dst < world; ++dst) {
      const int64_t lo = base[src] > new_start[dst] ? base[src] : new_start[dst];
      const int64_t hi = base[src + 1] < new_start[dst + 1] ? base[src + 1] : new_start[dst + 1];
      counts[(size_t)src * world + dst] = hi > lo ? hi - lo : 0;
    }
  return PA_OK;
}

int pa_dist_plan_check(int32_t world, const int64_t* new_start, const int64_t* cap, const int64_t* base, const int64_t* R_cur) {
  if (world < 1 || !new_start || ((base == nullptr) != (R_cur == nullptr))) return PA_EINVAL;
  if (new_start[world] >= (1ll << 32) - 4096) return PA_ECAPACITY;  // global slot indices are 32-bit
  int rc = PA_OK;
  for (int r = 0; r < world; ++r) {
    const int64_t n = new_start[r + 1] - new_start[r];
    if (n < 0) return PA_EINVAL;
    if (cap && n > cap[r]) return PA_ECAPACITY;  // capacity first: the same answer on every rank whatever the order of the defects
    if (cap && base) {  // theta > 0: what a rank receives is landed behind its R_cur parents in the current buffer
      const int64_t lo = base[r] > new_start[r] ? base[r] : new_start[r];
      const int64_t hi = base[r + 1] < new_start[r + 1] ? base[r + 1] : new_start[r + 1];
      const int64_t stay = hi > lo ? hi - lo : 0;
      if (R_cur[r] + (n - stay) > cap[r]) return PA_ECAPACITY;
    }
    if (n == 0) rc = PA_EEXTINCT;
  }
  return rc;
}

int pa_dist_capacity(pa_ctx* c, int64_t* cap) {
  if (!c || !cap) return PA_EINVAL;
  if (c->world < 1) return fail(c, PA_EINVAL, "pa_dist_capacity: not a shard");
  *cap = c->cap;
  return PA_OK;
}

int pa_dist_init(const pa_config* cfg, int32_t rank, int32_t world, pa_ctx** out) {
  if (!cfg || !out || world < 1 || rank < 0 || rank >= world || cfg->R0 < world) return PA_EINVAL;
  if (cfg->policy != PA_POLICY_BALANCED && world > BAL_PMAX) return PA_EINVAL;
  if (cfg->flags & PA_RESAMPLE_SYSTEMATIC) return PA_EINVAL;  // A4c's prefix sum would span the ranks (reading G30)
  pa_config local = *cfg;
  const int64_t first = balanced_start(cfg->R0, world, rank), last = balanced_start(cfg->R0, world, rank + 1);
  local.R0 = last - first;
  local.P = 1;
  local.policy = PA_POLICY_BALANCED;  // the device keeps one local partition; the policy acts between the ranks
  if (local.capacity == 0) local.capacity = (2 * ((cfg->R0 + world - 1) / world) + 4096 + 1023) / 1024 * 1024;
  int rc = init_common(&local, out, rank, world, cfg->R0, first);
  if (*out) {
    (*out)->cfg.policy = cfg->policy;  // for the rank-level plan
    (*out)->cfg.block = cfg->block;
    (*out)->cfg.maxexc = cfg->maxexc;
  }
  return rc;
}

uint64_t pa_dist_workspace_bytes(const pa_config* cfg, int32_t world) {
  if (!cfg || world < 1 || cfg->R0 < world) return 0;
  pa_config local = *cfg;
  local.R0 = (cfg->R0 + world - 1) / world;
  local.P = 1;
  local.policy = PA_POLICY_BALANCED;
  if (local.capacity == 0) local.capacity = (2 * ((cfg->R0 + world - 1) / world) + 4096 + 1023) / 1024 * 1024;
  Layout lo;
  if (!make_layout(&local, local.capacity, &lo, true)) return 0;
  return lo.total;
}

int pa_dist_begin(pa_ctx* c, double beta_next, int32_t theta, pa_dist_partial* mine) {
  if (!c || !mine) return PA_EINVAL;
  if (c->world < 1) return fail(c, PA_EINVAL, "pa_dist_begin: not a shard (use pa_dist_init)");
  if (c->dist_phase != 0) return fail(c, PA_EINVAL, "pa_dist_begin: a step is in flight");
  if (int rc = bind_device(c)) return rc;
  if (int rc = check_step_args(c, c->beta, beta_next, theta)) return rc;
  if ((uint64_t)c->steps + 1u >= (1ull << 28)) return fail(c, PA_EINVAL, "step counter would exceed 2^28");
  c->h_params[0] = make_params(c, c->beta, beta_next, theta);
  StepParams* d_params = c->dev<StepParams>(c->lo.params);
  CK(cudaMemcpyAsync(d_params, c->h_params, sizeof(StepParams), cudaMemcpyHostToDevice, c->stream));
  DevState* st = c->dev<DevState>(c->lo.state);
  const int n_desc = (int)((c->cap + SCAN_TILE - 1) / SCAN_TILE + 1);
  {
    Prof p(c, PA_K_Q_REDUCE);  // a shard: stops at the rank's own sum of weights
    launch(c, "k_q_reduce", k_q_reduce, c->red_grid, RED_THREADS, st, (const StepParams*)d_params,
           (const int32_t*)c->dev<int32_t>(c->lo.EM[0]), (const int32_t*)c->dev<int32_t>(c->lo.EM[1]), c->N,
           c->dev<double>(c->lo.red_partial), (double)c->g_R0, c->dev<unsigned long long>(c->lo.tile_desc), n_desc, tables(c), c->nearest);
  }
  if (int rc = sync_state(c)) return rc;
  mine->sumw = c->h_state->sumw;
  mine->R = c->R;
  c->dist_phase = 1;
  c->dist_theta = theta;
  c->dist_beta_next = beta_next;
  return PA_OK;
}

int pa_dist_resample(pa_ctx* c, const pa_dist_partial* all, int64_t* offspring) {
  if (!c || !all || !offspring) return PA_EINVAL;
  if (c->world < 1 || c->dist_phase != 1) return fail(c, PA_EINVAL, "pa_dist_resample: call pa_dist_begin first");
  if (int rc = bind_device(c)) return rc;
  double sumw = 0.0;  // the ranks' sums are added in rank order on every rank: all ranks get the same bits
  int64_t R = 0;
  for (int r = 0; r < c->world; ++r) {
    sumw += all[r].sumw;
    R += all[r].R;
  }
  if (all[c->rank].R != c->R) return fail(c, PA_EINVAL, "pa_dist_resample: all[rank] is not this rank's partial");
  DevState* st = c->dev<DevState>(c->lo.state);
  const StepParams* d_params = c->dev<StepParams>(c->lo.params);
  const LevelTables tb = tables(c);
  const int32_t *E0 = c->dev<int32_t>(c->lo.EM[0]), *E1 = c->dev<int32_t>(c->lo.EM[1]);
  {
    Prof p(c, PA_K_LEVELS_TAU);
    launch(c, "k_dist_tables", k_dist_tables, 1u, RED_THREADS, st, d_params, c->N, sumw, (double)R, (double)c->g_R0, tb, c->nearest);
  }
  {
    const bool keep = c->lo.n || c->lo.tau;
    ScanOut out;
    out.off = c->dev<uint32_t>(c->lo.off);
    out.n = c->lo.n ? c->dev<uint32_t>(c->lo.n) : nullptr;
    out.tau = c->lo.tau ? c->dev<double>(c->lo.tau) : nullptr;
    out.tile_desc = c->dev<unsigned long long>(c->lo.tile_desc);
    out.parent_of = c->dev<uint32_t>(c->lo.parent_of);
    out.tile_parent = c->dev<uint32_t>(c->lo.tile_parent);
    const int shift = copy_shift_for(c->cfg.L);
    const unsigned long long cap = (unsigned long long)c->cap;
    c->dist_lean = c->dist_theta > 0;
    c->dist_packed = false;
    if (c->dist_lean) out.parent_of = c->dev<uint32_t>(c->lo.dist_map);  // child -> parent map of the rank's own offspring
    const unsigned grid = scan_grid(c, c->dist_lean);
    Prof p(c, PA_K_POISSON_SCAN);
    launch_scan(c, keep, c->dist_lean, grid, st, E0, E1, tb, out, shift, cap);
  }
  // theta = 0: the rank's offspring, expanded in child order, into the spare buffer: the send side of the exchange.
  // theta > 0: nothing is expanded here; pa_dist_pack gathers only the slices that leave the rank, the sweep's load the rest.
  if (!c->dist_lean) launch_copy(c);
  CK(cudaMemcpyAsync(c->h_state, st, sizeof(DevState), cudaMemcpyDeviceToHost, c->stream));
  CK(cudaStreamSynchronize(c->stream));
  CK(cudaGetLastError());
  if (!c->launch_err.empty()) {  // a launch of this phase failed: report it now, not at some later synchronisation
    const std::string msg = "kernel launch failed: " + c->launch_err;
    c->launch_err.clear();
    return fail(c, PA_ECUDA, msg);
  }
  const DevState& hs = *c->h_state;
  // a rank without offspring is fine here (extinction is a property of the whole population: the plan reports it)
  if (hs.status == ST_CAPACITY) *offspring = -1;
  else *offspring = (int64_t)hs.Rnew;
  c->dist_T = (int64_t)hs.Rnew;
  c->dist_phase = 2;
  return PA_OK;
}

int pa_dist_pack(pa_ctx* c, const int64_t* T_all, int32_t* self_in_exchange) {
  if (!c || !T_all) return PA_EINVAL;
  if (c->world < 1 || c->dist_phase != 2) return fail(c, PA_EINVAL, "pa_dist_pack: call pa_dist_resample first");
  if (self_in_exchange) *self_in_exchange = c->dist_lean ? 0 : 1;
  if (!c->dist_lean) return PA_OK;  // theta = 0: pa_dist_resample has expanded everything, own share included
  if (int rc = bind_device(c)) return rc;
  const int W = c->world, me = c->rank;
  std::vector<int64_t> ns(W + 1), base(W + 1), counts((size_t)W * W);
  const int rc = pa_dist_exchange_plan(W, T_all, (int)c->cfg.policy, c->cfg.block, c->cfg.maxexc, ns.data(), base.data(), counts.data());
  if (rc != PA_OK) return fail(c, rc, rc == PA_EEXTINCT ? "population extinct (sum of offspring = 0)" : "a rank's offspring exceed its capacity");
  const int64_t T = base[me + 1] - base[me], n_new = ns[me + 1] - ns[me];
  if (T != c->dist_T) return fail(c, PA_EINVAL, "pa_dist_pack: T_all[rank] is not this rank's offspring total");
  auto clamp = [](int64_t x, int64_t lo, int64_t hi) { return x < lo ? lo : (x > hi ? hi : x); };
  const int64_t a = clamp(ns[me] - base[me], 0, T), b = clamp(ns[me + 1] - base[me], a, T);  // [a, b) stay
  const int64_t n_lo = clamp(base[me] - ns[me], 0, n_new), n_stay = b - a, n_recv = n_new - n_stay;
  if (n_new > c->cap || c->R + n_recv > c->cap)
    return fail(c, PA_ECAPACITY, "the rank's new share, or its parents plus what it receives, exceed its capacity (pa_dist_plan_check refuses this on all ranks)");
  const int64_t n_out = a + (T - b);
  if (n_out > 0) {
    const uint64_t words = (uint64_t)n_out * c->wrep;
    const unsigned grid = (unsigned)std::min<uint64_t>((words + 255) / 256, 148 * 16);
    launch(c, "k_dist_pack", k_dist_pack, grid, 256u, (const DevState*)c->dev<DevState>(c->lo.state), c->dev<uint32_t>(c->lo.spins[0]),
           c->dev<uint32_t>(c->lo.spins[1]), (const uint32_t*)c->dev<uint32_t>(c->lo.dist_map), (unsigned long long)a,
           (unsigned long long)b, (unsigned long long)T, c->wrep);
  }
  {
    const unsigned grid = (unsigned)std::min<uint64_t>(((uint64_t)n_new + 255) / 256, 148 * 8);
    launch(c, "k_dist_compose", k_dist_compose, grid ? grid : 1u, 256u, (const uint32_t*)c->dev<uint32_t>(c->lo.dist_map), c->dev<uint32_t>(c->lo.parent_of),
           (unsigned long long)n_new, (unsigned long long)n_lo, (unsigned long long)n_stay, (unsigned long long)a, (unsigned long long)c->R);
  }
  CK(cudaGetLastError());  // enqueued, not synchronised: the caller orders its exchange after cfg.stream
  c->dist_recv = n_recv;
  c->dist_packed = true;
  return PA_OK;
}

int pa_dist_buffers(pa_ctx* c, void** children, void** population) {
  if (!c) return PA_EINVAL;
  if (c->world < 1 || c->dist_phase != 2) return fail(c, PA_EINVAL, "pa_dist_buffers: no step in flight");
  const unsigned cur = c->h_state->cur;
  if (c->dist_lean && !c->dist_packed) return fail(c, PA_EINVAL, "pa_dist_buffers: call pa_dist_pack first (theta > 0)");
  if (children) *children = c->dev<char>(c->lo.spins[cur ^ 1u]);
  // theta = 0: the new population replaces the parents; theta > 0: what arrives is landed behind the R parents
  if (population) *population = c->dev<char>(c->lo.spins[cur]) + (c->dist_lean ? (size_t)c->R * (size_t)(c->N / 8) : 0);
  return PA_OK;
}

int pa_dist_new_count(pa_ctx* c, const int64_t* T_all, int64_t* count, int64_t* first_global_slot) {
  if (!c || !T_all) return PA_EINVAL;
  if (c->world < 1) return fail(c, PA_EINVAL, "pa_dist_new_count: not a shard");
  const int W = c->world;
  std::vector<int64_t> ns(W + 1), base(W + 1), counts((size_t)W * W);
  const int rc = pa_dist_exchange_plan(W, T_all, (int)c->cfg.policy, c->cfg.block, c->cfg.maxexc, ns.data(), base.data(), counts.data());
  if (rc != PA_OK) return fail(c, rc, rc == PA_EEXTINCT ? "population extinct (sum of offspring = 0)" : "a rank's offspring exceed its capacity");
  const int64_t n = ns[c->rank + 1] - ns[c->rank];
  if (count) *count = n;
  if (first_global_slot) *first_global_slot = ns[c->rank];
  if (n > c->cap) return fail(c, PA_ECAPACITY, "the rank's share of the new population exceeds its capacity");
  if (ns[W] >= (1ll << 32) - 4096) return fail(c, PA_ECAPACITY, "global population does not fit 32-bit slot indices");
  return PA_OK;
}

int pa_dist_abort(pa_ctx* c) {
  if (!c) return PA_EINVAL;
  if (c->world < 1) return fail(c, PA_EINVAL, "pa_dist_abort: not a shard");
  if (int rc = bind_device(c)) return rc;
  k_clear_status<<<1, 1, 0, c->stream>>>(c->dev<DevState>(c->lo.state));
  c->launches += 1;
  c->dist_phase = 0;
  c->attempt_failed = true;  // off / n / tau hold the dropped attempt: pa_tau / pa_counts refuse until the next commit
  return sync_state(c);
}

int pa_dist_finish(pa_ctx* c, const int64_t* T_all, pa_obs* local) {
  if (!c || !T_all) return PA_EINVAL;
  if (c->world < 1 || c->dist_phase != 2) return fail(c, PA_EINVAL, "pa_dist_finish: call pa_dist_resample first");
  if (int rc = bind_device(c)) return rc;
  int64_t n = 0, first = 0;
  // Both refusals below are reached only by a caller that skipped pa_dist_plan_check (which refuses them on EVERY rank
  // before the exchange).  Nothing has been committed: the step stays in flight and pa_dist_abort drops it.
  if (int rc = pa_dist_new_count(c, T_all, &n, &first)) {
    c->attempt_failed = true;
    return rc;
  }
  if (n < 1) {
    c->attempt_failed = true;
    return fail(c, PA_EEXTINCT, "this rank's share of the new population is empty (pa_dist_plan_check refuses such a plan on all ranks)");
  }
  DevState* st = c->dev<DevState>(c->lo.state);
  k_clear_status<<<1, 1, 0, c->stream>>>(st);  // a capacity flag of the local expansion cannot be pending here (plan refused it)
  k_dist_set_new<<<1, 1, 0, c->stream>>>(st, (unsigned long long)n, (unsigned)first);
  c->launches += 2;
  const StepParams& hp = c->h_params[0];
  if (c->dist_lean) {
    if (!c->dist_packed) {
      c->attempt_failed = true;
      return fail(c, PA_EINVAL, "pa_dist_finish: pa_dist_pack was not called for this step (theta > 0)");
    }
    // the sweep's load gathers the new population from the current buffer (own children from their parents, received
    // lattices from behind the parents) into the spare one, as in the one-GPU step; the commit flips the buffers
    launch_sweep(c, c->dist_theta, hp.T4, hp.T8, 2);
    launch_observe(c, c->dev<StepParams>(c->lo.params), 0, true);
  } else {
    launch_sweep(c, c->dist_theta, hp.T4, hp.T8, 3);  // in place: E, M only
    launch_observe(c, c->dev<StepParams>(c->lo.params), 2);
  }
  c->dist_phase = 0;
  if (int rc = sync_state(c)) {
    c->attempt_failed = true;
    return rc;
  }
  c->attempt_failed = false;
  if (local) return pa_observables(c, local);
  return PA_OK;
}

int pa_profile_read(pa_ctx* c, double* ms, int64_t* launches) {
  if (!c || !ms || !launches) return PA_EINVAL;
  for (int k = 0; k < PA_K_COUNT; ++k) {
    ms[k] = 0.0;
    launches[k] = 0;
  }
  CK(cudaStreamSynchronize(c->stream));
  for (EventPair& ep : c->ev_used) {
    float t = 0.f;
    CK(cudaEventElapsedTime(&t, ep.a, ep.b));
    ms[ep.kernel] += t;
    launches[ep.kernel] += 1;
    c->ev_free.push_back(ep);
  }
  c->ev_used.clear();
  return PA_OK;
}

int pa_launch_count(pa_ctx* c, int64_t* launches) {
  if (!c || !launches) return PA_EINVAL;
  *launches = c->launches;
  return PA_OK;
}

const char* pa_last_error(pa_ctx* c) { return c ? c->err.c_str() : "null context"; }

int pa_destroy(pa_ctx* c) {
  if (!c) return PA_EINVAL;
  cudaStreamSynchronize(c->stream);
  for (EventPair& ep : c->ev_used) { cudaEventDestroy(ep.a); cudaEventDestroy(ep.b); }
  for (EventPair& ep : c->ev_free) { cudaEventDestroy(ep.a); cudaEventDestroy(ep.b); }
  if (c->h_state) cudaFreeHost(c->h_state);
  if (c->h_params) cudaFreeHost(c->h_params);
  delete c;
  return PA_OK;
}

}  // extern "C"
