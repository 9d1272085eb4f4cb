"""Seeded synthetic workloads (BASELINE.json `configs`) and crafted populations for tests.

This module holds NO arithmetic of the method (no Philox, no energies, no weights): it only names shapes,
schedules and seeds, and draws generic random test data with numpy.  It is the one module that the
oracle-side tests and the CUDA-side tests both import; it imports neither of them.

The paper measures on no public dataset: its workload is itself a synthetic 2D Ising anneal (L=64, beta 0->1
in 200 steps, 20 480 replicas per GPU, theta in {1,10}).  The five configs below are
that workload's shapes.
"""
from dataclasses import dataclass

import numpy as np


@dataclass(frozen=True)
class Workload:
    name: str
    L: int          # lattice side, N = L*L spins, S = N/8 bytes per packed replica
    R0: int         # initial = target population R_beta0
    K: int          # number of temperature steps
    beta0: float    # inverse temperature the population is declared to be at
    beta_K: float   # final inverse temperature (uniform steps)
    theta: int      # MCMC sweeps per temperature step
    P: int          # logical partitions
    seed: int

    @property
    def N(self):
        return self.L * self.L

    @property
    def bytes_per_replica(self):
        return self.N // 8

    def beta(self, k):
        """inverse temperature after step k (k = 0..K); uniform schedule"""
        return self.beta0 + (self.beta_K - self.beta0) * k / self.K

    def scaled(self, R0, K=None):
        """same lattice/schedule at a reduced population (and optionally fewer steps of the same dbeta)"""
        K2 = self.K if K is None else K
        beta_K = self.beta0 + (self.beta_K - self.beta0) * K2 / self.K
        return Workload(self.name + "@R%d" % R0, self.L, R0, K2, self.beta0, beta_K, self.theta, self.P, self.seed)


# BASELINE.json configs[0..4]  (1-based names as in SURVEY.md section 8)
CONFIGS = {
    1: Workload("config1_L8_R1024", 8, 1 << 10, 100, 0.0, 1.0, 10, 1, 1),
    2: Workload("config2_L32_R65536", 32, 1 << 16, 200, 0.0, 1.0, 10, 1, 2),
    3: Workload("config3_L64_R2M", 64, 1 << 21, 100, 0.0, 0.5, 10, 148, 3),
    4: Workload("config4_L128_R1M", 128, 1 << 20, 500, 0.0, 0.6, 20, 148, 4),
    # resampling/redistribution stress: uniform random lattices DECLARED at beta=0.40, one step to 0.45, theta=0
    5: Workload("config5_resample_L32_R16M", 32, 1 << 24, 1, 0.40, 0.45, 0, 148, 5),
}

# the paper's own scalability task on 8 GPUs: L = 64, beta 0 -> 1 in K = 200 steps, 20 480 replicas
# per GPU, theta = 1; here the 8 GPUs are 8 logical partitions of one device (Fig. 1-2 shapes)
PAPER_TASK = Workload("paper_task_L64_8x20480", 64, 8 * 20480, 200, 0.0, 1.0, 1, 8, 6)


def random_packed_population(L, R, seed, p_up=0.5):
    """generic random bit lattices (R, N/32) uint32 for tests of set_spins / energy kernels; NOT the method's
    init (that one is Philox-keyed and implemented independently on both sides)."""
    rng = np.random.default_rng(seed)
    N = L * L
    bits = (rng.random((R, N)) < p_up).astype(np.uint8)
    by = np.packbits(bits, axis=1, bitorder="little")
    pad = (-by.shape[1]) % 4
    if pad:
        by = np.concatenate([by, np.zeros((R, pad), np.uint8)], axis=1)
    return np.ascontiguousarray(by).view(np.uint32).reshape(R, -1).copy()


def structured_population(L, R, seed):
    """mixture of ordered, striped, checkerboard, domain-wall and random lattices: spans the energy range
    (-2N .. +2N) so that reweighting produces strongly skewed copy counts; for parity tests."""
    rng = np.random.default_rng(seed)
    N = L * L
    yy, xx = np.divmod(np.arange(N), L)
    pats = [np.ones(N, np.uint8), np.zeros(N, np.uint8), ((xx + yy) & 1).astype(np.uint8),
            (yy & 1).astype(np.uint8), (xx & 1).astype(np.uint8), (yy < L // 2).astype(np.uint8),
            (xx < L // 3).astype(np.uint8)]
    out = np.zeros((R, N), np.uint8)
    for j in range(R):
        kind = rng.integers(0, len(pats) + 3)
        if kind < len(pats):
            b = pats[kind].copy()
            nflip = rng.integers(0, max(2, N // 16))
            b[rng.integers(0, N, nflip)] ^= 1
        else:
            b = (rng.random(N) < rng.choice([0.1, 0.5, 0.9])).astype(np.uint8)
        out[j] = b
    by = np.packbits(out, axis=1, bitorder="little")
    pad = (-by.shape[1]) % 4
    if pad:
        by = np.concatenate([by, np.zeros((R, pad), np.uint8)], axis=1)
    return np.ascontiguousarray(by).view(np.uint32).reshape(R, -1).copy()


# ---- second workload: the 2D +-J spin glass ----------------------------------
def bond_sample(L, seed, p_neg=0.5):
    """one disorder sample: (Jx, Jy), int8 arrays of N couplings +-1 in site order b = y*L + x; Jx[b] couples
    (x,y)-(x+1,y), Jy[b] couples (x,y)-(x,y+1), periodic.  P(J = -1) = p_neg (0.5: the symmetric +-J model)."""
    rng = np.random.default_rng(seed)
    N = L * L
    Jx = np.where(rng.random(N) < p_neg, -1, 1).astype(np.int8)
    Jy = np.where(rng.random(N) < p_neg, -1, 1).astype(np.int8)
    return Jx, Jy


def mattis_bonds(L, seed):
    """gauge transform of the ferromagnet: J_ij = eps_i eps_j for random eps = +-1 (no frustration); returns
    (Jx, Jy, eps).  Every quantity of the ferromagnet maps onto this sample by sigma -> eps * sigma."""
    rng = np.random.default_rng(seed)
    eps = np.where(rng.random((L, L)) < 0.5, -1, 1).astype(np.int8)
    Jx = (eps * np.roll(eps, -1, axis=1)).astype(np.int8).reshape(-1)
    Jy = (eps * np.roll(eps, -1, axis=0)).astype(np.int8).reshape(-1)
    return Jx, Jy, eps.reshape(-1)


def pack_pm1(a):
    """+-1 values (..., n) with n a multiple of 32 -> little-endian bit string as uint32 words, bit 1 <-> +1 (layout C2)"""
    a = np.asarray(a)
    bits = (a > 0).astype(np.uint8)
    by = np.packbits(bits, axis=-1, bitorder="little")
    return np.ascontiguousarray(by).view(np.uint32).copy()
