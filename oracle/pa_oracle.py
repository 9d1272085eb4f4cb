"""Population-annealing oracle driver -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Sequences the plain C routines of oracle/pa_oracle.c in the paper's order:
reweight (eq. 3, 4) -> Poisson resample -> place offspring / balance partitions -> theta MCMC
sweeps -> observables, and keeps the free-energy recursion of eq. 5 (reading G1).
Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  It never imports the CUDA package.
"""
import ctypes as C
import math
import os

import numpy as np

from . import build as _build

_lib = None


def lib():
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(path)
        u32p, i32p, f64p, u64p, i8p = (C.POINTER(C.c_uint32), C.POINTER(C.c_int32), C.POINTER(C.c_double),
                                       C.POINTER(C.c_uint64), C.POINTER(C.c_int8))
        sig = {
            "orc_max_threads": (C.c_int, []),
            "orc_set_threads": (None, [C.c_int]),
            "orc_philox4x32_10": (None, [u32p, u32p, u32p]),
            "orc_words_per_replica": (C.c_int64, [C.c_int]),
            "orc_energy_mag": (None, [C.c_int, C.c_int64, u32p, i32p, i32p]),
            "orc_init_population": (None, [C.c_int, C.c_int64, C.c_uint64, u32p]),
            "orc_q": (C.c_double, [C.c_int64, i32p, C.c_double]),
            "orc_q_by_levels": (C.c_double, [C.c_int64, i32p, C.c_double, C.c_int]),
            "orc_tau": (None, [C.c_int64, i32p, C.c_double, C.c_double, f64p]),
            "orc_expneg": (C.c_double, [C.c_double]),
            "orc_uniform_resample": (C.c_double, [C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint64]),
            "orc_poisson": (C.c_uint32, [C.c_double, C.c_uint64, C.c_uint32, C.c_uint32]),
            "orc_poisson_counts": (None, [C.c_int64, f64p, C.c_double, C.c_uint64, C.c_uint32, u32p]),
            "orc_nearest": (C.c_uint32, [C.c_double, C.c_uint64, C.c_uint32, C.c_uint32]),
            "orc_nearest_counts": (None, [C.c_int64, f64p, C.c_double, C.c_uint64, C.c_uint32, u32p]),
            "orc_systematic_uniform": (C.c_uint32, [C.c_uint64, C.c_uint32]),
            "orc_systematic_counts": (None, [C.c_int64, f64p, C.c_double, C.c_uint64, C.c_uint32, u32p]),
            "orc_overlap": (C.c_double, [C.c_int64, i32p, C.c_double]),
            "orc_adaptive_dbeta": (C.c_double, [C.c_int64, i32p, C.c_double, C.c_double, C.c_int]),
            "orc_exclusive_scan": (C.c_int64, [C.c_int64, u32p, u32p]),
            "orc_copy": (None, [C.c_int, C.c_int64, u32p, u32p, u32p, i32p, i32p, u32p, i32p, i32p]),
            "orc_parent_of": (None, [C.c_int64, u32p, u32p, C.c_int64, u32p]),
            "orc_partition_table": (None, [C.c_int64, C.c_int, u32p]),
            "orc_partition_stats": (C.c_int64, [C.c_int64, u32p, u32p, C.c_int, u32p, u32p, u32p]),
            "orc_policy_counts": (C.c_int64, [C.c_int, u32p, C.c_int, C.c_uint32, C.c_uint32, u32p]),
            "orc_starts_from_counts": (None, [C.c_int, u32p, u32p]),
            "orc_thresholds": (None, [C.c_double, u32p, u32p]),
            "orc_sweeps": (None, [C.c_int, C.c_int64, C.c_int64, u32p, C.c_uint64, C.c_uint32, C.c_int,
                                  C.c_uint32, C.c_uint32]),
            "orc_sweeps_slots": (None, [C.c_int, C.c_int64, u32p, u32p, C.c_uint64, C.c_uint32, C.c_int,
                                        C.c_uint32, C.c_uint32]),
            "orc_moment_sums": (None, [C.c_int64, i32p, i32p, u64p]),
            "orc_energy_int8": (C.c_int32, [C.c_int, i8p]),
            "orc_energy_mag_J": (None, [C.c_int, C.c_int64, u32p, i8p, i8p, i32p, i32p]),
            "orc_energy_int8_J": (C.c_int32, [C.c_int, i8p, i8p, i8p]),
            "orc_sweeps_J": (None, [C.c_int, C.c_int64, C.c_int64, u32p, C.c_uint64, C.c_uint32, C.c_int,
                                    C.c_uint32, C.c_uint32, i8p, i8p]),
            "orc_sweeps_slots_J": (None, [C.c_int, C.c_int64, u32p, u32p, C.c_uint64, C.c_uint32, C.c_int,
                                          C.c_uint32, C.c_uint32, i8p, i8p]),
            "orc_overlap_hist": (None, [C.c_int, C.c_int64, u32p, u64p]),
            "orc_pack": (None, [C.c_int, i8p, u32p]),
            "orc_unpack": (None, [C.c_int, u32p, i8p]),
        }
        for name, (res, args) in sig.items():
            fn = getattr(L, name)
            fn.restype = res
            fn.argtypes = args
        _lib = L
    return _lib


def _p(a, ct):
    return a.ctypes.data_as(C.POINTER(ct))


def _c(a, dtype):
    a = np.ascontiguousarray(a, dtype=dtype)
    return a


# ------------------------------------------------------------------------------------------------
# thin function wrappers (one C call each)
# ------------------------------------------------------------------------------------------------
def max_threads():
    return int(lib().orc_max_threads())


def set_threads(n):
    lib().orc_set_threads(int(n))


def philox4x32_10(ctr, key):
    c = _c(ctr, np.uint32)
    k = _c(key, np.uint32)
    out = np.zeros(4, np.uint32)
    lib().orc_philox4x32_10(_p(c, C.c_uint32), _p(k, C.c_uint32), _p(out, C.c_uint32))
    return out


def words_per_replica(L):
    return int(lib().orc_words_per_replica(int(L)))


def init_population(L, R, seed):
    packed = np.zeros((R, words_per_replica(L)), np.uint32)
    lib().orc_init_population(L, R, C.c_uint64(seed), _p(packed, C.c_uint32))
    return packed


def _bonds(L, bonds):
    """(Jx, Jy): int8 arrays of N couplings +-1, site order b = y*L + x (oracle/pa_oracle.c section D1)"""
    Jx, Jy = (_c(np.asarray(b).reshape(-1), np.int8) for b in bonds)
    assert Jx.shape[0] == L * L and Jy.shape[0] == L * L and set(np.unique(np.concatenate([Jx, Jy]))) <= {-1, 1}
    return Jx, Jy


def energy_mag(L, packed, bonds=None):
    packed = _c(packed, np.uint32)
    R = packed.shape[0]
    E = np.zeros(R, np.int32)
    M = np.zeros(R, np.int32)
    if bonds is None:
        lib().orc_energy_mag(L, R, _p(packed, C.c_uint32), _p(E, C.c_int32), _p(M, C.c_int32))
    else:
        Jx, Jy = _bonds(L, bonds)
        lib().orc_energy_mag_J(L, R, _p(packed, C.c_uint32), _p(Jx, C.c_int8), _p(Jy, C.c_int8), _p(E, C.c_int32),
                               _p(M, C.c_int32))
    return E, M


def overlap_hist(L, packed):
    """hist[(q + N) / 2] over the pairs (j, j + R // 2) (oracle/pa_oracle.c section D1, reading G28)"""
    packed = _c(packed, np.uint32)
    hist = np.zeros(L * L + 1, np.uint64)
    lib().orc_overlap_hist(L, packed.shape[0], _p(packed, C.c_uint32), _p(hist, C.c_uint64))
    return hist


def q_ratio(E, dbeta):
    E = _c(E, np.int32)
    return float(lib().orc_q(E.shape[0], _p(E, C.c_int32), float(dbeta)))


def q_ratio_by_levels(E, dbeta, N):
    E = _c(E, np.int32)
    return float(lib().orc_q_by_levels(E.shape[0], _p(E, C.c_int32), float(dbeta), int(N)))


def tau_weights(E, dbeta, Q):
    E = _c(E, np.int32)
    tau = np.zeros(E.shape[0], np.float64)
    lib().orc_tau(E.shape[0], _p(E, C.c_int32), float(dbeta), float(Q), _p(tau, C.c_double))
    return tau


def expneg(mu):
    return float(lib().orc_expneg(float(mu)))


def uniform_resample(seed, step, j, c):
    return float(lib().orc_uniform_resample(C.c_uint64(seed), int(step), int(j), C.c_uint64(c)))


def poisson(lam, seed, step, j):
    return int(lib().orc_poisson(float(lam), C.c_uint64(seed), int(step), int(j)))


def poisson_counts(tau, scale, seed, step):
    tau = _c(tau, np.float64)
    n = np.zeros(tau.shape[0], np.uint32)
    lib().orc_poisson_counts(tau.shape[0], _p(tau, C.c_double), float(scale), C.c_uint64(seed), int(step),
                             _p(n, C.c_uint32))
    return n


RULE_POISSON, RULE_NEAREST, RULE_SYSTEMATIC = 0, 1, 2
ADAPTIVE_ITERS = 40  # bisection steps of the adaptive temperature step (reading G25)


def nearest(lam, seed, step, j):
    return int(lib().orc_nearest(float(lam), C.c_uint64(seed), int(step), int(j)))


def nearest_counts(tau, scale, seed, step):
    tau = _c(tau, np.float64)
    n = np.zeros(tau.shape[0], np.uint32)
    lib().orc_nearest_counts(tau.shape[0], _p(tau, C.c_double), float(scale), C.c_uint64(seed), int(step), _p(n, C.c_uint32))
    return n


def systematic_uniform(seed, step):
    return int(lib().orc_systematic_uniform(C.c_uint64(seed), int(step)))


def systematic_counts(tau, scale, seed, step):
    tau = _c(tau, np.float64)
    n = np.zeros(tau.shape[0], np.uint32)
    lib().orc_systematic_counts(tau.shape[0], _p(tau, C.c_double), float(scale), C.c_uint64(seed), int(step), _p(n, C.c_uint32))
    return n


def overlap(E, dbeta):
    E = _c(E, np.int32)
    return float(lib().orc_overlap(E.shape[0], _p(E, C.c_int32), float(dbeta)))


def adaptive_dbeta(E, target, dbeta_max, iters=ADAPTIVE_ITERS):
    E = _c(E, np.int32)
    return float(lib().orc_adaptive_dbeta(E.shape[0], _p(E, C.c_int32), float(target), float(dbeta_max), int(iters)))


def exclusive_scan(n):
    n = _c(n, np.uint32)
    off = np.zeros(n.shape[0] + 1, np.uint32)
    total = int(lib().orc_exclusive_scan(n.shape[0], _p(n, C.c_uint32), _p(off, C.c_uint32)))
    return off, total


def copy_population(L, n, off, src, Esrc, Msrc, Rnew):
    src = _c(src, np.uint32)
    dst = np.zeros((Rnew, src.shape[1]), np.uint32)
    Ed = np.zeros(Rnew, np.int32)
    Md = np.zeros(Rnew, np.int32)
    n = _c(n, np.uint32)
    off = _c(off, np.uint32)
    Esrc = _c(Esrc, np.int32)
    Msrc = _c(Msrc, np.int32)
    lib().orc_copy(L, n.shape[0], _p(n, C.c_uint32), _p(off, C.c_uint32), _p(src, C.c_uint32),
                   _p(Esrc, C.c_int32), _p(Msrc, C.c_int32), _p(dst, C.c_uint32), _p(Ed, C.c_int32),
                   _p(Md, C.c_int32))
    return dst, Ed, Md


def parent_of(n, off, Rnew):
    n = _c(n, np.uint32)
    off = _c(off, np.uint32)
    parent = np.zeros(Rnew, np.uint32)
    lib().orc_parent_of(n.shape[0], _p(n, C.c_uint32), _p(off, C.c_uint32), Rnew, _p(parent, C.c_uint32))
    return parent


def partition_table(Rpop, P):
    ps = np.zeros(P + 1, np.uint32)
    lib().orc_partition_table(int(Rpop), int(P), _p(ps, C.c_uint32))
    return ps


def partition_stats(n, off, P, old_start, new_start):
    n = _c(n, np.uint32)
    off = _c(off, np.uint32)
    old_start = _c(old_start, np.uint32)
    new_start = _c(new_start, np.uint32)
    stats = np.zeros((P, 4), np.uint32)
    moved = int(lib().orc_partition_stats(n.shape[0], _p(n, C.c_uint32), _p(off, C.c_uint32), int(P),
                                          _p(old_start, C.c_uint32), _p(new_start, C.c_uint32),
                                          _p(stats, C.c_uint32)))
    return stats, moved


POLICY_BALANCED, POLICY_MAIN, POLICY_NAIVE, POLICY_NONE = 0, 1, 2, 3


def policy_counts(born, policy, block=1024, maxexc=1):
    """cnt_p of every partition after redistribution under `policy` (A6b); also the number of block moves"""
    born = _c(born, np.uint32)
    cnt = np.zeros(born.shape[0], np.uint32)
    moves = int(lib().orc_policy_counts(born.shape[0], _p(born, C.c_uint32), int(policy), int(block), int(maxexc),
                                        _p(cnt, C.c_uint32)))
    return cnt, moves


def starts_from_counts(cnt):
    cnt = _c(cnt, np.uint32)
    start = np.zeros(cnt.shape[0] + 1, np.uint32)
    lib().orc_starts_from_counts(cnt.shape[0], _p(cnt, C.c_uint32), _p(start, C.c_uint32))
    return start


def thresholds(beta):
    t4 = C.c_uint32(0)
    t8 = C.c_uint32(0)
    lib().orc_thresholds(float(beta), C.byref(t4), C.byref(t8))
    return int(t4.value), int(t8.value)


def sweeps(L, packed, seed, step, theta, T4, T8, first=0, count=None, bonds=None):
    """In place on `packed` (R, wpr) uint32, slots first..first+count-1."""
    assert packed.dtype == np.uint32 and packed.flags.c_contiguous
    if count is None:
        count = packed.shape[0] - first
    if bonds is None:
        lib().orc_sweeps(L, int(first), int(count), _p(packed, C.c_uint32), C.c_uint64(seed), int(step), int(theta),
                         int(T4), int(T8))
    else:
        Jx, Jy = _bonds(L, bonds)
        lib().orc_sweeps_J(L, int(first), int(count), _p(packed, C.c_uint32), C.c_uint64(seed), int(step), int(theta),
                           int(T4), int(T8), _p(Jx, C.c_int8), _p(Jy, C.c_int8))


def sweeps_slots(L, slots, packed_list, seed, step, theta, T4, T8, bonds=None):
    """In place on packed_list[i] (the lattice living in population slot slots[i])."""
    assert packed_list.dtype == np.uint32 and packed_list.flags.c_contiguous
    slots = _c(slots, np.uint32)
    if bonds is None:
        lib().orc_sweeps_slots(L, slots.shape[0], _p(slots, C.c_uint32), _p(packed_list, C.c_uint32), C.c_uint64(seed),
                               int(step), int(theta), int(T4), int(T8))
    else:
        Jx, Jy = _bonds(L, bonds)
        lib().orc_sweeps_slots_J(L, slots.shape[0], _p(slots, C.c_uint32), _p(packed_list, C.c_uint32),
                                 C.c_uint64(seed), int(step), int(theta), int(T4), int(T8), _p(Jx, C.c_int8),
                                 _p(Jy, C.c_int8))


def moment_sums(E, M):
    E = _c(E, np.int32)
    M = _c(M, np.int32)
    out = np.zeros(10, np.uint64)
    lib().orc_moment_sums(E.shape[0], _p(E, C.c_int32), _p(M, C.c_int32), _p(out, C.c_uint64))
    vals = [int(out[2 * i]) | (int(out[2 * i + 1]) << 64) for i in range(5)]
    if vals[0] >= 1 << 127:  # sum E is signed
        vals[0] -= 1 << 128
    return {"sum_E": vals[0], "sum_E2": vals[1], "sum_absM": vals[2], "sum_M2": vals[3], "sum_M4": vals[4]}


def energy_int8(L, s, bonds=None):
    s = _c(s, np.int8)
    if bonds is None:
        return int(lib().orc_energy_int8(L, _p(s, C.c_int8)))
    Jx, Jy = _bonds(L, bonds)
    return int(lib().orc_energy_int8_J(L, _p(s, C.c_int8), _p(Jx, C.c_int8), _p(Jy, C.c_int8)))


def pack(L, s):
    s = _c(s, np.int8)
    w = np.zeros(words_per_replica(L), np.uint32)
    lib().orc_pack(L, _p(s, C.c_int8), _p(w, C.c_uint32))
    return w


def unpack(L, words):
    words = _c(words, np.uint32)
    s = np.zeros(L * L, np.int8)
    lib().orc_unpack(L, _p(words, C.c_uint32), _p(s, C.c_int8))
    return s


def default_capacity(R0):
    """Slots per buffer when the caller passes capacity=0 (DESIGN.md boundary): R' ~ Poisson(R0), so
    R0 + max(1024, 16*ceil(sqrt(R0))) rounded up to a multiple of 1024 is a 16-sigma margin."""
    ceil_sqrt = math.isqrt(R0 - 1) + 1 if R0 > 0 else 0
    cap = R0 + max(1024, 16 * ceil_sqrt)
    return (cap + 1023) // 1024 * 1024


class OracleError(Exception):
    pass


class OraclePA:
    """State + step sequencing.  Notation follows the paper: R (current population R_beta_i), R0
    (R_beta_0), Q (eq. 3), tau (eq. 4), theta (MCMC sweeps per temperature)."""

    def __init__(self, L, R0, P=1, seed=0, beta0=0.0, capacity=0, spins=None, policy=POLICY_BALANCED, block=1024,
                 maxexc=1, rule=RULE_POISSON, bonds=None):
        self.rule = int(rule)
        self.bonds = bonds  # None: the Ising ferromagnet of eq. (6); (Jx, Jy): the +-J model (section D1)
        self.L, self.N, self.R0, self.P, self.seed = int(L), int(L) * int(L), int(R0), int(P), int(seed)
        self.capacity = int(capacity) if capacity else default_capacity(self.R0)
        self.policy, self.block, self.maxexc = int(policy), int(block), int(maxexc)
        self.beta = float(beta0)
        self.step_no = 0
        # A1: initial population; or a caller-supplied population (test hook)
        self.spins = init_population(self.L, self.R0, self.seed) if spins is None else _c(spins, np.uint32).copy()
        self.R = self.spins.shape[0]
        self.E, self.M = energy_mag(self.L, self.spins, self.bonds)
        # eq. 5 (reading G1): ln Z(beta_i) = ln Omega + sum_l ln Q(beta_{l-1}, beta_l), ln Omega = N ln 2
        self.ln_omega = self.N * math.log(2.0)
        self.sum_lnQ = 0.0
        self.last_Q = float("nan")
        self.part_start = partition_table(self.R, self.P)
        self.last = {}

    @property
    def lnZ(self):
        return self.ln_omega + self.sum_lnQ

    # ---- a1-a6 -----------------------------------------------------------------------------
    def resample(self, beta_next, tau_override=None):
        """Reweight + Poisson resample + offspring placement + partition table.
        tau_override: lock-step parity mode -- draw the counts from the GPU's tau (north_star:
        "copy counts must be bit-exact when the oracle is driven from the GPU's tau")."""
        dbeta = float(beta_next) - self.beta
        if not (abs(dbeta) * 2 * self.N < 700.0):
            raise OracleError("exp range (reading G11)")
        step = self.step_no + 1
        Q = q_ratio(self.E, dbeta)                                   # eq. 3
        tau = tau_weights(self.E, dbeta, Q)                          # eq. 4
        scale = float(self.R0) / float(self.R)                       # reading G2
        tau_used = tau if tau_override is None else _c(tau_override, np.float64)
        if self.rule == RULE_SYSTEMATIC:
            n = systematic_counts(tau_used, scale, self.seed, step)  # A4c
        elif self.rule == RULE_NEAREST:
            n = nearest_counts(tau_used, scale, self.seed, step)     # A4b
        else:
            n = poisson_counts(tau_used, scale, self.seed, step)    # A4
        off, Rnew = exclusive_scan(n)                                # A5
        if Rnew > self.capacity:
            raise OracleError("capacity")
        if Rnew == 0:
            raise OracleError("extinct")
        if self.policy == POLICY_BALANCED:
            new_start = partition_table(Rnew, self.P)                # A6
        else:                                                        # A6b: main / naive / none
            born = np.diff(off[self.part_start].astype(np.int64)).astype(np.uint32)
            cnt, _ = policy_counts(born, self.policy, self.block, self.maxexc)
            new_start = starts_from_counts(cnt)
        stats, moved = partition_stats(n, off, self.P, self.part_start, new_start)
        spins, E, M = copy_population(self.L, n, off, self.spins, self.E, self.M, Rnew)
        self.last = {"Q": Q, "tau": tau, "n": n, "off": off, "Rnew": Rnew, "part_start": new_start,
                     "part_stats": stats, "moved": moved, "dbeta": dbeta, "R_parents": self.R}
        self.spins, self.E, self.M, self.R = spins, E, M, Rnew
        self.part_start = new_start
        self.sum_lnQ += math.log(Q)                                  # eq. 5
        self.last_Q = Q
        self.beta = float(beta_next)
        self.step_no = step
        return self.last

    # ---- a7, a8 ----------------------------------------------------------------------------
    def equilibrate(self, theta):
        if theta > 0:
            T4, T8 = thresholds(self.beta)
            sweeps(self.L, self.spins, self.seed, self.step_no, theta, T4, T8, bonds=self.bonds)
            self.E, self.M = energy_mag(self.L, self.spins, self.bonds)

    def step(self, beta_next, theta, tau_override=None):
        info = self.resample(beta_next, tau_override)
        self.equilibrate(theta)
        return info

    def adaptive_beta(self, target, dbeta_max):
        """A9: the next inverse temperature for a histogram overlap `target`"""
        return self.beta + adaptive_dbeta(self.E, target, dbeta_max)

    def observables(self):
        s = moment_sums(self.E, self.M)
        R = float(self.R)
        s.update({"R": self.R, "mean_E": s["sum_E"] / R, "mean_E2": s["sum_E2"] / R, "mean_absM": s["sum_absM"] / R,
                  "mean_M2": s["sum_M2"] / R, "mean_M4": s["sum_M4"] / R})
        return s
