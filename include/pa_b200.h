/*
 * pa_b200.h -- C ABI of the B200-native population-annealing (PA) hot path for the 2D Ising model.
 *
 * What is computed is defined by arxiv 2006.00561 and the readings in DESIGN.md:
 *   reweight   Q(beta,beta') = sum_j exp[-(beta'-beta) E_j] / R            PAPER.md:46  eq. (3), :94
 *              tau_j = exp[-(beta'-beta) E_j] / Q                           PAPER.md:51  eq. (4)
 *   resample   n_j ~ Poisson(tau_j * R0/R), offspring = exact copies
 *   redistribute  new population balanced over P logical partitions
 *   equilibrate   theta MCMC (checkerboard Metropolis) sweeps at beta'
 *   observe    population sums of E, E^2, |M|, M^2, M^4; ln Z recursion     PAPER.md:62, :66 eq. (5)
 *   model      H = -(J/2) sum' sigma sigma', J = 1, periodic L x L          PAPER.md:76-80 eq. (6)
 *              (or, after pa_set_bonds, the +-J spin glass on the same lattice  PAPER.md:213)
 *
 * Conventions
 *   - plain C, no exceptions; every function returns PA_OK (0) or a negative pa_status;
 *     pa_last_error(ctx) gives a message for the last failure on that context.
 *   - pointers marked DEVICE are CUDA device pointers, HOST are host pointers; getters take a flag
 *     saying which kind `dst` is.  All device work is issued on cfg.stream.
 *   - ownership: the CALLER owns the device workspace and the stream (PyTorch allocates both); the library
 *     owns only the host-side pa_ctx (and a few bytes of pinned host memory inside it).  pa_destroy never
 *     frees the workspace.
 *   - packed lattice layout ("C2" in DESIGN.md): a replica is an N = L*L bit little-endian string, spin (x,y)
 *     is bit b = y*L + x, stored in uint32 word b>>5 at bit b&31, bit 1 <-> sigma = +1; slot i of the
 *     population starts at byte i * N/8.
 *   - one context per host thread; a context is bound to the device that was current in pa_init.
 *   - there is NO CPU fallback: without a CUDA device pa_init returns PA_ECUDA.
 */
#ifndef PA_B200_H
#define PA_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct pa_ctx pa_ctx; /* opaque, host side, library owned */

typedef enum {
  PA_OK = 0,
  PA_EINVAL = -1,    /* bad argument (L, P, theta, NaN beta, |dbeta|*2N >= 700, getter without its KEEP flag) */
  PA_ENOMEM = -2,    /* workspace smaller than pa_workspace_bytes(cfg) */
  PA_ECAPACITY = -3, /* resampled population R' > capacity: step NOT committed, population unchanged */
  PA_EEXTINCT = -4,  /* R' = 0: step NOT committed, population unchanged */
  PA_ECUDA = -5      /* CUDA runtime error (message in pa_last_error) */
} pa_status;

enum {
  PA_KEEP_TAU = 1u,    /* materialise tau_j of every step (8 B per parent) for pa_tau */
  PA_KEEP_COUNTS = 2u, /* materialise n_j of every step (4 B per parent) for pa_counts(n != NULL) */
  PA_PROFILE = 4u,     /* record CUDA events around every kernel (pa_profile_read); the events between the kernels
                          keep a kernel's blocks from being placed while its predecessor drains */
  PA_PROFILE_SPAN = 8u, /* record only the PA_K_RESAMPLE_SPAN pair around a1-a6 of every step */
  PA_RESAMPLE_NEAREST = 16u, /* copy counts n_j = floor(lambda_j) + [u_j > 1 - frac(lambda_j)] (nearest integers) instead of
                                Poisson(lambda_j): one of the modifications PAPER.md:54 points to; A4b */
  PA_RESAMPLE_SYSTEMATIC = 32u /* systematic resampling (A4c): one keyed uniform per step, copy counts from the exact
                                  64-bit cumulative sum of floor(lambda_j 2^32): the population stays at R0.  Excludes
                                  PA_RESAMPLE_NEAREST; not available for pa_dist_init (PA_EINVAL) */
};

/* Redistribution policies (A6b, readings G21-G23).  The children are in parent order and a
 * partition is a contiguous range of them; a policy decides the counts cnt_p.  It changes the partition table and the
 * diagnostics only -- population, weights and copy counts do not depend on it. */
enum {
  PA_POLICY_BALANCED = 0, /* cnt_p = floor(R'/P) + (p < R' mod P): counts differ by <= 1 replica */
  PA_POLICY_MAIN = 1,     /* the paper's main algorithm: blocks of `block` replicas move from the largest excess to the
                             largest shortage until every partition is within `maxexc` blocks of its balanced count */
  PA_POLICY_NAIVE = 2,    /* the paper's naive algorithm: every partition pools floor(born_p / 2) replicas -- a number
                             proportional to its offspring -- and the pool is dealt back evenly */
  PA_POLICY_NONE = 3      /* no redistribution: cnt_p = born_p */
};

typedef struct {
  int32_t L;        /* lattice side: 8, 16, 32, 64 or 128 */
  int32_t P;        /* logical partitions, >= 1 (148 = one per B200 SM); <= 1024 unless policy = PA_POLICY_BALANCED */
  int64_t R0;       /* initial = target population R_beta0, 1 <= R0 < 2^31 */
  int64_t capacity; /* slots per population buffer; 0 => R0 + max(1024, 16*ceil(sqrt(R0))) rounded up to 1024 */
  uint64_t seed;    /* Philox key */
  double beta0;     /* inverse temperature the initial population is declared to be at (uniform init is exact for 0) */
  void* workspace;  /* DEVICE memory, caller owned, 256-byte aligned, >= pa_workspace_bytes(cfg) */
  uint64_t workspace_bytes;
  void* stream;     /* cudaStream_t, caller owned (NULL = legacy default stream) */
  uint32_t flags;   /* PA_KEEP_TAU | PA_KEEP_COUNTS | PA_PROFILE | PA_PROFILE_SPAN | PA_RESAMPLE_NEAREST or _SYSTEMATIC */
  uint32_t policy;  /* PA_POLICY_*: how the new population is divided over the P partitions (default 0 = balanced) */
  uint32_t block;   /* PA_POLICY_MAIN: replicas per block (0 => 1024) */
  uint32_t maxexc;  /* PA_POLICY_MAIN: window in blocks (0 => 1) */
} pa_config;

/* population sums after the last committed step (or after pa_init / pa_set_spins); 128-bit integers as {lo, hi} */
typedef struct {
  int64_t R;            /* population size the sums run over */
  int64_t sum_E;        /* sum_j E_j                     (|sum| < 2^63 for every supported size) */
  uint64_t sum_E2[2];   /* sum_j E_j^2 */
  uint64_t sum_absM[2]; /* sum_j |M_j| */
  uint64_t sum_M2[2];   /* sum_j M_j^2 */
  uint64_t sum_M4[2];   /* sum_j M_j^4                   (exceeds 2^64 for L = 128, R = 2^20) */
  double mean_E, mean_E2, mean_absM, mean_M2, mean_M4; /* sums / R in fp64 */
} pa_obs;

/* per-partition diagnostics of the last step, in the paper's vocabulary */
typedef struct {
  uint32_t cnt;  /* replicas the partition holds after redistribution */
  uint32_t born; /* offspring of the parents that lived in this partition (what it would hold without redistribution) */
  uint32_t maxg; /* excess   max(0, born - cnt) */
  uint32_t minl; /* shortage max(0, cnt - born) */
} pa_part_stats;

/* kernels of one pa_step, in launch order (indices of pa_profile_read arrays) */
enum {
  PA_K_LEVELS_W = 0, /* (w_e = exp(-dbeta e) per level is tabulated inside PA_K_Q_REDUCE: reports 0 launches) */
  PA_K_Q_REDUCE,     /* eq. 3: fp64 warp-shuffle reduction, Q, ln Q; its last block: eq. 4 per level + Poisson tables */
  PA_K_LEVELS_TAU,   /* (run by the last block of PA_K_Q_REDUCE: reports 0 launches) */
  PA_K_POISSON_SCAN, /* Poisson copy counts + single-pass exclusive scan + child -> parent map */
  PA_K_BALANCE,      /* partition table + diagnostics: run by the last block of PA_K_OBSERVE, reports 0 launches */
  PA_K_COPY,         /* replica redistribution: gather copy (theta = 0 only; with theta > 0 the lattices are gathered
                        by PA_K_SWEEP's load and this reports 0 launches) */
  PA_K_SWEEP,        /* theta checkerboard Metropolis sweeps + E, M */
  PA_K_OBSERVE,      /* population sums + commit of the step */
  PA_K_RESAMPLE_SPAN, /* not a kernel: elapsed time on cfg.stream from the start of PA_K_Q_REDUCE to the end of PA_K_COPY
                         (theta = 0) or of PA_K_POISSON_SCAN (theta > 0): a1-a6 as one span */
  PA_K_COUNT
};

/* Bytes of device workspace needed for cfg (L, R0, capacity, P, flags are read).  0 on invalid cfg. */
uint64_t pa_workspace_bytes(const pa_config* cfg);

/* a0. Create a context and the initial population: R0 replicas of uniform +-1 spins from Philox (seed),
 * E_j, M_j, ln Omega = N ln 2.  Synchronises the stream before returning. */
int pa_init(const pa_config* cfg, pa_ctx** out);

/* a1-a8. One temperature step beta -> beta_next with theta >= 0 sweeps.  Synchronous: returns after the step's
 * kernels finished and its status was read back.  On PA_ECAPACITY / PA_EEXTINCT the population, beta, step
 * counter and ln Z (and pa_log_Z's last_Q) are unchanged.  pa_step is pa_run with K = 1: one stream synchronisation
 * and one 264-byte read-back of the device state per call; queue whole schedules with pa_run to avoid both. */
int pa_step(pa_ctx* ctx, double beta_next, int32_t theta);

/* The asynchronous form of the step that SURVEY.md 8(b) describes (pa_step is its K = 1 case with a synchronisation).
 * K steps beta_k = betas[k] (HOST array of K doubles), all launched back to back with ONE synchronisation at the
 * end; stops committing at the first failing step (later steps are no-ops) and reports it.  *steps_done (may be
 * NULL) receives the number of committed steps. */
int pa_run(pa_ctx* ctx, const double* betas, int32_t K, int32_t theta, int32_t* steps_done);

/* Adaptive temperature step (A9): *beta_next = beta + the largest dbeta in (0, dbeta_max] whose
 * histogram overlap alpha(dbeta) = (1/R) sum_j min(1, tau_j(dbeta)) is >= target_overlap (40 bisection steps on
 * [0, dbeta_max]).  Only proposes the temperature: follow with pa_step(*beta_next, theta).  Synchronises. */
int pa_adaptive_beta(pa_ctx* ctx, double target_overlap, double dbeta_max, double* beta_next);

int pa_population(pa_ctx* ctx, int64_t* R);
int pa_beta(pa_ctx* ctx, double* beta, int64_t* steps);
/* work counter: sum over all committed steps of the resampled population size R' (replica-steps); the number of
 * spin-flip attempts of a run with constant theta is theta * N * (difference of this counter) */
int pa_totals(pa_ctx* ctx, int64_t* replica_steps);

/* E_j (and M_j) of slots 0..n-1 of the current population, slot order.  n <= R.  M may be NULL. */
int pa_energies(pa_ctx* ctx, int32_t* E, int32_t* M, int64_t n, int dst_on_device);

/* eq. 5 (reading G1): *lnZ = N ln 2 + sum_lnQ; *last_Q = Q of the last committed step. NULLs allowed. */
int pa_log_Z(pa_ctx* ctx, double* lnZ, double* sum_lnQ, double* last_Q);

int pa_observables(pa_ctx* ctx, pa_obs* out);

/* ---- parity / debug getters --------------------------------------------------------------------------- */
/* packed lattices of slots first..first+count-1 (count * N/32 uint32 words) */
int pa_spins(pa_ctx* ctx, uint32_t* dst, int64_t first, int64_t count, int dst_on_device);
/* tau_j of the LAST step's parents, j = 0..n-1, n <= number of parents (needs PA_KEEP_TAU).  PA_EINVAL after a step
 * that was not committed (PA_ECAPACITY / PA_EEXTINCT) until the next committed step: the arrays then hold the failed
 * attempt.  Same for pa_counts. */
int pa_tau(pa_ctx* ctx, double* dst, int64_t n, int dst_on_device);
/* copy counts n_j (needs PA_KEEP_COUNTS; may be NULL) and exclusive offsets off_j, j = 0..n_parents (off has
 * n_parents+1 entries, off[n_parents] = R') of the LAST step */
int pa_counts(pa_ctx* ctx, uint32_t* n, uint32_t* off, int64_t n_parents, int dst_on_device);
/* number of parents of the last step (population size before it) */
int pa_parents(pa_ctx* ctx, int64_t* n_parents);
/* partition table of the current population (HOST, P+1 entries) and the last step's diagnostics (HOST, P
 * entries, may be NULL); *moved (may be NULL) = children whose partition differs from their parent's */
int pa_partitions(pa_ctx* ctx, uint32_t* part_start, pa_part_stats* stats, int64_t* moved);
/* acceptance thresholds used by the last step with theta > 0 */
int pa_thresholds(pa_ctx* ctx, uint32_t* T4, uint32_t* T8);
/* test hook (parity only): while enabled, every later step uses T4, T8 as its acceptance thresholds instead of
 * floor(2^32 exp(-4 beta')), floor(2^32 exp(-8 beta')) (C4) -- lets a test reach u == T and the extreme
 * thresholds 0 and 2^32 - 1, which no temperature produces on demand.  pa_thresholds reports the values used. */
int pa_debug_set_thresholds(pa_ctx* ctx, int enable, uint32_t T4, uint32_t T8);
/* test hook: replace the population by R packed lattices (R <= capacity); recomputes E, M, sums, partitions;
 * beta, step counter and ln Z are kept */
int pa_set_spins(pa_ctx* ctx, const uint32_t* src, int64_t R, int src_on_device);

/* ---- second Hamiltonian: the 2D +-J spin glass (D1) ---------- */
/* Replace eq. (6) by H = - sum_<ij> J_ij sigma_i sigma_j with one sample of couplings J_ij = +-1 shared by all
 * replicas.  Jx, Jy: HOST arrays of N/32 uint32 words each, bit layout C2 (bit b = y*L + x, bit 1 <-> J = +1):
 * Jx couples (x,y)-(x+1,y), Jy couples (x,y)-(x,y+1), indices modulo L.  Both NULL: back to the ferromagnet.  Only
 * before the first temperature step (PA_EINVAL afterwards); recomputes E_j and the population sums, synchronises.
 * Everything else (weights, resampling, redistribution, acceptance thresholds, keying) is unchanged: E = 2u - 2N with
 * u = number of unsatisfied bonds, E = 2 * (#negative bonds) mod 4.  On a multi-GPU shard every rank sets the same sample. */
int pa_set_bonds(pa_ctx* ctx, const uint32_t* Jx, const uint32_t* Jy);
/* Order parameter of the spin glass: overlap q = sum_i sigma_i^a sigma_i^b of replica j and replica
 * j + floor(R/2), j < floor(R/2) (reading G28); hist (HOST, N+1 entries): hist[(q + N) / 2] = number of pairs.
 * Works for either Hamiltonian; synchronises. */
int pa_overlap_hist(pa_ctx* ctx, uint64_t* hist);

/* ---- for callers that must not allocate: one call that creates nothing ---------------------------------- */
/* Every other entry point needs a pa_ctx (pa_init pins host memory) and a workspace the caller has allocated.  This one
 * needs neither, for users who cannot allocate when they want the order-parameter histogram: a hook running while
 * something else (a framework's caching allocator, another simulation) holds all of the GPU's memory; a monitoring loop
 * that must not stall the device (cudaFree synchronises it, cudaMalloc can); code that is handed a device pointer and a
 * stream and nothing else.  It calls no cudaMalloc / cudaFree / cudaHostAlloc and no routine that does.
 *
 * Computes what pa_overlap_hist computes (D1, reading G28), on lattices the CALLER holds:
 *   spins  DEVICE, R packed lattices of L x L spins in layout C2 (R * L*L/32 uint32 words), on the current GPU, read only
 *   hist   L*L + 1 uint64 entries, HOST (hist_on_device = 0) or DEVICE (1), overwritten:
 *          hist[(q + N) / 2] = number of pairs (j, j + floor(R/2)), j < floor(R/2), with overlap q
 *   stream cudaStream_t of the current GPU (NULL = legacy default stream); all device work is issued on it
 * HOST hist: returns after the result has arrived (synchronises the stream).  DEVICE hist: returns after enqueueing.
 *
 * The 64-bit accumulation bins -- scratch the context path keeps in its workspace -- are a fixed array inside the
 * library image: 131 328 bytes (128*128 + 1 counters, padded) on every GPU that loads the library, held until the process
 * exits.  Limit: L <= PA_STATIC_MAX_L; a larger L returns PA_EINVAL ("lattice too large for the static scratch").
 * Also PA_EINVAL: L not in {8,16,32,64,128}, R outside [0, 2^31), NULL pointers, spins not device memory of the
 * current GPU.  PA_ECUDA: a CUDA call failed.  pa_static_last_error() has the message (per host thread).
 *
 * The array is shared by all calls on a GPU and keeps the previous call's counts; each call clears the bins it uses
 * first.  Calls whose GPU work may overlap (different streams without an ordering between them, concurrent host
 * threads) race on it and return garbage; calls on one stream or separated by a synchronisation are safe.
 * The first call on each GPU looks up the array's device address (cudaGetSymbolAddress, with that GPU current), which
 * can make the CUDA runtime load the library's device code: make that first call early, before any stream capture
 * begins.  Later calls on that GPU reuse the address. */
#define PA_STATIC_MAX_L 128
int pa_overlap_hist_static(const uint32_t* spins, int32_t L, int64_t R, uint64_t* hist, int hist_on_device, void* stream);
const char* pa_static_last_error(void);

/* ---- multi-GPU: partitioned redistribution, one rank = one partition -------- */
/* The population is sharded over `world` ranks in global slot order: rank r owns the contiguous global slots
 * [start_r, start_{r+1}).  Every random number is keyed by the GLOBAL replica index, so the ranks together compute
 * exactly what one context with the whole population computes (up to the rounding of Q: the ranks' weight sums are
 * added in rank order).  A step is four calls with three small exchanges in between, which the CALLER performs (NCCL
 * through torch.distributed in paper_2006_00561_b200/dist.py; plain copies when the ranks are emulated on one device):
 *
 *   pa_dist_begin     local sum of weights                                  -> all-gather of pa_dist_partial
 *   pa_dist_resample  Q over all ranks, local Poisson counts + scan, the local offspring expanded in child order
 *                                                                           -> all-gather of the offspring totals T_r
 *   pa_dist_exchange_plan  (pure host function) global child offsets, new partition table under cfg.policy with
 *                     born_p = T_p (the paper's per-node offspring count), and the slice every rank sends to every other
 *   pa_dist_plan_check     (pure host function) every rank's share fits / is not empty, judged alike on every rank
 *   pa_dist_pack      theta > 0: gather the children that leave the rank into the send buffer
 *                                                                           -> all-to-all-v of lattices (contiguous slices)
 *   pa_dist_finish    theta sweeps of the new local population (theta > 0: gathered by the sweep's load), E, M, sums, commit
 *
 * Because global child order is source-rank order, the slices a rank receives are contiguous in its new buffer in source
 * order: the all-to-all-v writes straight into the population buffer (pa_dist_buffers), nothing is unpacked. */
typedef struct {
  double sumw; /* sum over the rank's replicas of exp[-(beta'-beta) E_j] */
  int64_t R;   /* the rank's current population */
} pa_dist_partial;

/* cfg.R0 = GLOBAL target population; cfg.capacity = slots per buffer of THIS rank (0 => twice the balanced share + 4096,
 * rounded up to 1024); cfg.P is ignored (partition = rank; <= 1024 ranks unless policy = balanced); cfg.policy / block /
 * maxexc govern the rank-level plan.  Creates the rank's share of the initial population (global balanced table). */
int pa_dist_init(const pa_config* cfg, int32_t rank, int32_t world, pa_ctx** out);
/* bytes of device workspace a rank needs for cfg (as given to pa_dist_init) */
uint64_t pa_dist_workspace_bytes(const pa_config* cfg, int32_t world);
int pa_dist_begin(pa_ctx* ctx, double beta_next, int32_t theta, pa_dist_partial* mine);
/* all: `world` entries in rank order (HOST).  *offspring = T_rank, or -1 if the rank's offspring exceed its capacity. */
int pa_dist_resample(pa_ctx* ctx, const pa_dist_partial* all, int64_t* offspring);
/* Pure host function, no CUDA: T = offspring totals in rank order; new_start[world+1] = global child index where each
 * rank's new range starts; base[world+1] = global child index where each rank's offspring start;
 * counts[src * world + dst] = children rank src sends to rank dst (its own share included).  PA_EEXTINCT if sum T = 0. */
int pa_dist_exchange_plan(int32_t world, const int64_t* T, int32_t policy, uint32_t block, uint32_t maxexc,
                          int64_t* new_start, int64_t* base, int64_t* counts);
/* Pure host function, no CUDA: may the plan be carried out?  new_start as written by pa_dist_exchange_plan; cap[r] = slots
 * per buffer of rank r in rank order (pa_dist_capacity, gathered together with the offspring totals; NULL = do not check).
 * PA_ECAPACITY if some rank's new share exceeds that rank's capacity (policy main can leave a rank up to block - 1
 * replicas above its balanced count) or the population outgrows 32-bit slot indices; PA_EEXTINCT if some rank's new share
 * is empty (policy none with a rank without offspring, or fewer children than ranks): a shard cannot be empty.  Every
 * rank evaluates this on the same gathered numbers BEFORE the exchange, so all ranks refuse the step or none does;
 * after a refusal every rank calls pa_dist_abort.  base (as written by the plan) and R_cur (the ranks' current populations,
 * known from the first all-gather) are given for a step with theta > 0 (both NULL for theta = 0): such a step lands what a
 * rank receives behind its parents, so R_cur[r] + (new share - children that stay) must fit cap[r] too. */
int pa_dist_plan_check(int32_t world, const int64_t* new_start, const int64_t* cap, const int64_t* base, const int64_t* R_cur);
/* slots per buffer of this rank (cfg.capacity as resolved by pa_dist_init) */
int pa_dist_capacity(pa_ctx* ctx, int64_t* cap);
/* Between the plan and the exchange.  theta > 0 (the lean step): nothing was expanded by pa_dist_resample; the rank's own
 * children that stay on the rank are gathered straight from their parents by the sweep's load in pa_dist_finish (as in
 * the one-GPU step), and this call gathers ONLY the children that leave the rank (a prefix for lower ranks, a suffix for
 * higher ranks; a few per cent near beta_c) into the send buffer, in destination order, and writes the gather map of the
 * new population.  *self_in_exchange = 0: the rank's own share is NOT part of the send and receive buffers.
 * theta = 0: no-op, *self_in_exchange = 1 (pa_dist_resample has expanded all offspring; the own share is copied by the
 * caller like any other slice).  The two small kernels are ENQUEUED on cfg.stream, not waited for: an exchange issued on
 * another stream (or by another library) must be ordered after cfg.stream by the caller (stream wait, event, or a
 * synchronisation).  PA_ECAPACITY if the plan does not fit (pa_dist_plan_check says so on every rank beforehand). */
int pa_dist_pack(pa_ctx* ctx, const int64_t* T_all, int32_t* self_in_exchange);
/* DEVICE pointers of the step in flight, valid between pa_dist_pack and pa_dist_finish: children = send side (slices in
 * destination order), population = receive side (slices in source order).  theta = 0: all offspring in child order / the
 * whole new population.  theta > 0: only what leaves the rank / only what arrives (own share absent on both sides). */
int pa_dist_buffers(pa_ctx* ctx, void** children, void** population);
/* T_all as given to the plan.  PA_ECAPACITY / PA_EEXTINCT if the rank's new share exceeds its capacity / is empty: check
 * BEFORE exchanging, on every rank for every rank, with pa_dist_plan_check -- a refusal here comes after the other ranks
 * have exchanged and would leave them committed while this one is not (the step stays in flight: pa_dist_abort).
 * local (may be NULL) receives the rank's population sums. */
int pa_dist_finish(pa_ctx* ctx, const int64_t* T_all, pa_obs* local);
/* the rank's share of the new population under the plan (and its first global slot); PA_ECAPACITY if it does not fit */
int pa_dist_new_count(pa_ctx* ctx, const int64_t* T_all, int64_t* count, int64_t* first_global_slot);
/* drop the step in flight on this rank (the plan was refused, or another rank failed): nothing was committed; pa_tau and
 * pa_counts return PA_EINVAL until the next committed step */
int pa_dist_abort(pa_ctx* ctx);

/* ---- profiling (PA_PROFILE) --------------------------------------------------------------------------- */
/* Sum of CUDA-event durations (ms) and number of launches per kernel since the last call; synchronises.
 * Both arrays have PA_K_COUNT entries (HOST). */
int pa_profile_read(pa_ctx* ctx, double* ms, int64_t* launches);
/* total number of kernels this context has launched since pa_init (all kernels, profiled or not) */
int pa_launch_count(pa_ctx* ctx, int64_t* launches);

const char* pa_last_error(pa_ctx* ctx);
int pa_destroy(pa_ctx* ctx); /* frees the host context only */

#ifdef __cplusplus
}
#endif
#endif /* PA_B200_H */
