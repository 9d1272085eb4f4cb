"""GPU parity (-m gpu): the CUDA path, called through the C ABI, against the CPU oracle on the same seeded inputs.

Bar (BASELINE.json north_star): spins, E, M, copy counts, offsets, R', partition tables and
integer moment sums BIT-EXACT; Q, tau, ln Z to relative 1e-12.  Lock-step: each step the oracle computes its own
Q / tau (compared at 1e-12) and then draws the counts from the GPU's tau array, so that every integer that
follows is compared exactly.
"""
import ctypes as C
import math
import os

import numpy as np
import pytest

from oracle import pa_oracle as orc
from paper_2006_00561_b200 import inputs

import philox_ref

pytestmark = pytest.mark.gpu

RTOL = 1e-12  # north_star: "Q, tau and ln Z must agree to a relative error of 1e-12 in fp64"


def _binding():
    from paper_2006_00561_b200 import binding
    return binding


def rel(a, b):
    return abs(a - b) / max(abs(b), 1e-300)


def make_pair(L, R0, P, seed, beta0=0.0, capacity=0, spins=None, policy=0, block=1024, maxexc=1, rule=0, bonds=None):
    b = _binding()
    gpu = b.PopulationAnnealer(L, R0, P=P, seed=seed, beta0=beta0, capacity=capacity,
                               flags=b.PA_KEEP_TAU | b.PA_KEEP_COUNTS | {0: 0, 1: b.PA_RESAMPLE_NEAREST, 2: b.PA_RESAMPLE_SYSTEMATIC}[rule], policy=policy,
                               block=block, maxexc=maxexc)
    if spins is not None:
        gpu.set_spins(spins)
    if bonds is not None:  # second Hamiltonian: +-J couplings (Jx, Jy) as int8 arrays in site order
        gpu.set_bonds(inputs.pack_pm1(bonds[0]), inputs.pack_pm1(bonds[1]))
    ora = orc.OraclePA(L, R0, P=P, seed=seed, beta0=beta0, capacity=capacity, spins=spins, policy=policy, block=block,
                       maxexc=maxexc, rule=rule, bonds=bonds)
    return gpu, ora


def compare_population(gpu, ora, what=""):
    assert gpu.R == ora.R, what
    assert np.array_equal(gpu.spins(), ora.spins), what + " spins"
    E, M = gpu.energies()
    assert np.array_equal(E, ora.E), what + " E"
    assert np.array_equal(M, ora.M), what + " M"
    og, oo = gpu.observables(), ora.observables()
    for k in ["R", "sum_E", "sum_E2", "sum_absM", "sum_M2", "sum_M4"]:
        assert og[k] == oo[k], (what, k, og[k], oo[k])
    for k in ["mean_E", "mean_E2", "mean_absM", "mean_M2", "mean_M4"]:
        assert rel(og[k], oo[k]) <= 1e-15 or abs(og[k] - oo[k]) <= 1e-12, (what, k)


def lockstep(gpu, ora, betas, theta, sweep_slots=None):
    """sweep_slots=None: full-population sweep parity; else an int: number of hash-selected slots checked."""
    L = ora.L
    for k, beta in enumerate(betas, 1):
        parents_before = ora.R
        spins_before = ora.spins
        gpu.step(beta, theta)
        tau_gpu = gpu.tau()
        info = ora.resample(beta, tau_override=tau_gpu)
        lz = gpu.log_Z()
        # fp64 quantities
        assert rel(lz["last_Q"], info["Q"]) <= RTOL, (k, lz["last_Q"], info["Q"])
        assert np.all(np.abs(tau_gpu - info["tau"]) <= RTOL * np.abs(info["tau"])), k
        assert rel(lz["lnZ"], ora.lnZ) <= RTOL, (k, lz["lnZ"], ora.lnZ)
        # integers
        assert gpu.parents() == parents_before
        n, off = gpu.counts()
        assert np.array_equal(n, info["n"]), "step %d: copy counts" % k
        assert np.array_equal(off, info["off"]), "step %d: offsets" % k
        assert gpu.R == info["Rnew"]
        ps, st, moved = gpu.partitions()
        assert np.array_equal(ps, info["part_start"]) and np.array_equal(st, info["part_stats"]), k
        assert moved == info["moved"], k
        if theta > 0:
            assert gpu.thresholds() == orc.thresholds(beta)
        if sweep_slots is None:
            ora.equilibrate(theta)
            compare_population(gpu, ora, "step %d" % k)
        else:
            # a1-a6 on the full population: children are exact copies of their parents, in parent order.
            # Sweeps: hash-selected slots, each swept alone by the oracle (depends only on lattice, slot, seed, step)
            # plus, always, the edges of the sweep kernels' blocks (16 / 64 replicas per block) and the partly filled last one
            rng = np.random.default_rng(1000 + k)
            edges = [s_ for s_ in (0, 15, 16, 63, 64) if s_ < ora.R] + list(range(max(0, ora.R - 17), ora.R))
            slots = np.unique(np.concatenate([rng.integers(0, ora.R, sweep_slots), np.asarray(edges, np.int64)])).astype(np.uint32)
            before = ora.spins[slots].copy()
            parent = orc.parent_of(info["n"], info["off"], info["Rnew"])
            assert np.array_equal(before, spins_before[parent[slots]])
            if theta > 0:
                T4, T8 = orc.thresholds(beta)
                orc.sweeps_slots(L, slots, before, ora.seed, ora.step_no, theta, T4, T8, bonds=ora.bonds)
            got = gpu.spins()
            assert np.array_equal(got[slots], before), "step %d: sampled sweeps" % k
            if theta == 0:  # no sweeps: the whole redistributed population is comparable
                assert np.array_equal(got, ora.spins), "step %d: redistribution" % k
            # adopt the GPU population for the next step, after checking E/M of ALL replicas against the oracle's
            # energy function (plain definition) -- keeps the oracle in lock-step without sweeping everything
            E, M = gpu.energies()
            Eo, Mo = orc.energy_mag(L, got, ora.bonds)
            assert np.array_equal(E, Eo) and np.array_equal(M, Mo)
            ora.spins, ora.E, ora.M = got, Eo, Mo
            og, oo = gpu.observables(), ora.observables()
            for key in ["R", "sum_E", "sum_E2", "sum_absM", "sum_M2", "sum_M4"]:
                assert og[key] == oo[key], (k, key)


# ---------------------------------------------------------------------------------------------------
# C3: Philox -- product device function == cuRAND's curand_Philox4x32_10 == oracle == big-int writing
# ---------------------------------------------------------------------------------------------------
def test_philox_product_vs_curand_vs_oracle():
    import torch
    path = os.path.join(os.path.dirname(__file__), "cuda", "libphilox_check.so")
    if not os.path.exists(path):
        pytest.skip("tests/cuda/libphilox_check.so not built (run __graft_entry__.build())")
    lib = C.CDLL(path)
    n = 1 << 20
    rng = np.random.default_rng(2024)
    ctr = rng.integers(0, 2 ** 32, (n, 4), dtype=np.uint64).astype(np.uint32)
    key = rng.integers(0, 2 ** 32, (n, 2), dtype=np.uint64).astype(np.uint32)
    ctr[0], key[0] = 0, 0
    ctr[1], key[1] = 0xFFFFFFFF, 0xFFFFFFFF
    d = lambda a: torch.from_numpy(a.view(np.int32)).cuda()
    dc, dk = d(ctr), d(key)
    o1 = torch.zeros(n * 4, dtype=torch.int32, device="cuda")
    o2 = torch.zeros(n * 4, dtype=torch.int32, device="cuda")
    vp = C.c_void_p
    lib.philox_check.argtypes = [vp, vp, vp, vp, C.c_int]
    assert lib.philox_check(dc.data_ptr(), dk.data_ptr(), o1.data_ptr(), o2.data_ptr(), n) == 0
    a = o1.cpu().numpy().view(np.uint32).reshape(n, 4)
    b = o2.cpu().numpy().view(np.uint32).reshape(n, 4)
    assert np.array_equal(a, b)  # product == cuRAND on 2^20 random (ctr, key)
    for i in list(range(64)) + [n - 1]:
        assert a[i].tolist() == orc.philox4x32_10(ctr[i], key[i]).tolist() == philox_ref.philox4x32_10(ctr[i], key[i])


# ---------------------------------------------------------------------------------------------------
# a0 init, a8 energies
# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("L,R0", [(8, 1000), (16, 777), (32, 2049), (64, 515), (128, 130)])
def test_init_population_parity(L, R0):
    gpu, ora = make_pair(L, R0, P=3, seed=0x0123456789ABCDEF + L)
    compare_population(gpu, ora, "init L=%d" % L)
    assert rel(gpu.log_Z()["lnZ"], L * L * math.log(2)) < 1e-15
    ps, _, _ = gpu.partitions()
    assert np.array_equal(ps, orc.partition_table(R0, 3))


@pytest.mark.parametrize("L", [8, 16, 32, 64, 128])
def test_set_spins_energy_magnetisation(L):
    R = 300
    pop = inputs.structured_population(L, R, seed=L)
    gpu, ora = make_pair(L, R, P=1, seed=1, spins=pop)
    compare_population(gpu, ora, "set_spins L=%d" % L)
    E, _ = gpu.energies()
    assert E.min() < -1.5 * L * L and E.max() > 1.5 * L * L  # ordered and checkerboard-like lattices are in the mixture


# ---------------------------------------------------------------------------------------------------
# lock-step parity, whole step, every supported L
# ---------------------------------------------------------------------------------------------------
def test_config1_full_lockstep():
    wl = inputs.CONFIGS[1]
    gpu, ora = make_pair(wl.L, wl.R0, wl.P, wl.seed)
    compare_population(gpu, ora, "init")
    lockstep(gpu, ora, [wl.beta(k) for k in range(1, wl.K + 1)], wl.theta)
    exact = 128.715437337408418  # Kaufman L=8, beta=1 (tests/golden/ising_exact.json)
    assert abs(gpu.log_Z()["lnZ"] - exact) < 0.2


@pytest.mark.parametrize("L,R0,P,K,theta,dbeta", [
    (16, 3000, 5, 12, 3, 0.04),
    (32, 4096, 1, 16, 10, 0.03),     # config 2 shape, reduced population, coarser schedule crossing beta_c
    (64, 2048, 148, 8, 4, 0.06),      # config 3 shape
    (128, 600, 148, 5, 2, 0.02),      # config 4 shape (|dbeta|*2N < 700, reading G11)
])
def test_reduced_configs_lockstep(L, R0, P, K, theta, dbeta):
    gpu, ora = make_pair(L, R0, P, seed=L + 11)
    lockstep(gpu, ora, [dbeta * k for k in range(1, K + 1)], theta)


def test_ragged_population_sizes_and_theta1():
    # sizes around tile boundaries of the scan (2048), the copy (1024) and a warp
    for R0 in [1, 31, 33, 1023, 1025, 2047, 2049, 4097]:
        gpu, ora = make_pair(32, R0, P=7, seed=R0)
        lockstep(gpu, ora, [0.02, 0.05, 0.2], 1)


def test_skewed_resampling_heavy_parents():
    # structured population + a large dbeta: tau spans many decades, heavy parents (lambda >> 32) use the
    # warp-cooperative chunk loop; dead parents come in long runs
    L, R = 32, 20000
    pop = inputs.random_packed_population(L, R, seed=5)          # E ~ 0
    ordered = inputs.structured_population(L, 64, seed=6)         # a few lattices with E down to -2N
    where = np.random.default_rng(7).choice(R, 64, replace=False)
    pop[where] = ordered
    pop[5000:5300] = inputs.random_packed_population(L, 300, seed=8, p_up=0.5) ^ np.uint32(0x55555555)
    gpu, ora = make_pair(L, R, P=148, seed=55, beta0=0.3, spins=pop, capacity=40960)
    gpu.step(0.3 + 0.004, 0)
    tau = gpu.tau()
    info = ora.resample(0.3 + 0.004, tau_override=tau)
    n, off = gpu.counts()
    assert tau.max() > 100 and (info["n"] == 0).mean() > 0.5  # really skewed
    assert info["n"].max() > 64
    assert np.array_equal(n, info["n"]) and np.array_equal(off, info["off"])
    assert rel(gpu.log_Z()["last_Q"], info["Q"]) <= RTOL
    compare_population(gpu, ora, "skewed")
    ps, st, moved = gpu.partitions()
    assert np.array_equal(ps, info["part_start"]) and np.array_equal(st, info["part_stats"]) and moved == info["moved"]
    # a second step with sweeps from the skewed population
    lockstep(gpu, ora, [0.32], 2)


@pytest.mark.parametrize("L,R", [(64, 3000), (128, 1500), (16, 5000)])
def test_wide_level_window_fallback_paths(L, R):
    """crafted populations spanning -2N..+2N: the occupied level window is wider than the shared-memory tables
    (k_q_reduce evaluates exp per replica beyond 2048 levels; k_poisson_scan mixes cached and uncached levels), then
    narrows again after resampling -- every path must give the oracle's bits"""
    spins = inputs.structured_population(L, R, seed=100 + L)
    gpu, ora = make_pair(L, R, P=5, seed=9, beta0=0.2, spins=spins, capacity=4 * R)
    dbeta = 0.25 * 700.0 / (2 * L * L) if L >= 64 else 0.01   # large enough to skew the counts, within |dbeta| 2N < 700
    lockstep(gpu, ora, [0.2 + dbeta, 0.2 + 1.5 * dbeta, 0.2 + 1.6 * dbeta], 1)


def test_config5_reduced_resample_only():
    wl = inputs.CONFIGS[5].scaled(1 << 17)
    gpu, ora = make_pair(wl.L, wl.R0, wl.P, wl.seed, beta0=wl.beta0)
    lockstep(gpu, ora, [wl.beta_K], 0)
    n, _ = gpu.counts()
    assert n.max() >= 32 and (n == 0).mean() > 0.5  # the skew config 5 is meant to have


# ---------------------------------------------------------------------------------------------------
# full-size configs in the launch configuration bench.py times
# ---------------------------------------------------------------------------------------------------
def test_config2_full_size_first_steps():
    wl = inputs.CONFIGS[2]
    gpu, ora = make_pair(wl.L, wl.R0, wl.P, wl.seed)
    compare_population(gpu, ora, "init")
    lockstep(gpu, ora, [wl.beta(k) for k in range(1, 4)], wl.theta)


def test_config2_full_size_whole_schedule_in_three_stretches():
    """SURVEY.md 8(c) parity protocol, config 2: the FULL population (65 536 replicas: the launch shape of
    k_sweep_small<32,.,8> that bench.py times) compared after every step of three stretches of its own 200-step schedule --
    the first 20 steps, 15 steps across beta_c (0.405 -> 0.475), and the last 30 down to beta = 1.0, where nearly every
    site asks for a uniform and rejects.  Between the stretches the schedule is run with pa_run and the oracle adopts the
    population (its E, M recomputed and compared).  65 lock-step steps ~ 110 s of oracle time on 16 cores."""
    wl = inputs.CONFIGS[2]
    gpu, ora = make_pair(wl.L, wl.R0, wl.P, wl.seed)
    lockstep(gpu, ora, [wl.beta(k) for k in range(1, 21)], wl.theta)
    for k_from, k_to in ((80, 95), (170, 200)):
        done = gpu.beta_steps()[1]
        assert gpu.run([wl.beta(k) for k in range(done + 1, k_from + 1)], wl.theta) == k_from - done
        adopt(gpu, ora)
        lockstep(gpu, ora, [wl.beta(k) for k in range(k_from + 1, k_to + 1)], wl.theta)
    beta, steps = gpu.beta_steps()
    assert steps == wl.K == 200 and abs(beta - 1.0) < 1e-12
    assert gpu.observables()["mean_E"] / wl.N < -1.99           # ordered phase reached
    assert abs(gpu.log_Z()["lnZ"] / wl.N - inputs_exact_lnz_per_spin(32, 1.0)) < 2e-4


def inputs_exact_lnz_per_spin(L, beta):
    """ln Z / N of the L x L torus from the golden file written by tests/golden/make_ising_exact.py (Kaufman's formula)"""
    import json
    data = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "ising_exact.json")))
    return float(data["lnZ"]["L%d_beta%g" % (L, beta)]) / (L * L)


def test_config3_full_population_step_near_beta_c():
    """SURVEY.md 8(c) parity protocol, config 3: ONE step of its own dbeta = 0.005 schedule with the WHOLE population of
    2^21 replicas swept by the oracle and compared (spins, E, M, sums) -- step 88 (beta 0.435 -> 0.44, the critical region,
    where the population fluctuates most): every one of the 131 072 blocks of the k_sweep<64> launch that
    bench.py times, not a sample of slots.  ~ 215 s of oracle time on 16 cores."""
    wl = inputs.CONFIGS[3]
    gpu, ora = make_pair(wl.L, wl.R0, wl.P, wl.seed)
    assert gpu.run([wl.beta(k) for k in range(1, 88)], wl.theta) == 87
    adopt(gpu, ora)
    lockstep(gpu, ora, [wl.beta(88)], wl.theta)
    assert abs(gpu.beta_steps()[0] - 0.44) < 1e-12


def test_config3_full_size_sampled():
    wl = inputs.CONFIGS[3]
    gpu, ora = make_pair(wl.L, wl.R0, wl.P, wl.seed)
    compare_population(gpu, ora, "init")
    # coarse steps (|dbeta|*2N < 700, reading G11) up to the critical region, then two paper-sized steps
    lockstep(gpu, ora, [0.08, 0.16, 0.24, 0.32, 0.40, 0.435, 0.44], wl.theta, sweep_slots=4096)
    ps, st, _ = gpu.partitions()
    cnt = np.diff(ps.astype(np.int64))
    assert len(cnt) == 148 and cnt.max() - cnt.min() <= 1


def test_config4_full_size_sampled():
    wl = inputs.CONFIGS[4]
    gpu, ora = make_pair(wl.L, wl.R0, wl.P, wl.seed)
    lockstep(gpu, ora, [0.02, 0.04, 0.0412], wl.theta, sweep_slots=1024)


def test_config5_full_size():
    wl = inputs.CONFIGS[5]
    gpu, ora = make_pair(wl.L, wl.R0, wl.P, wl.seed, beta0=wl.beta0)
    lockstep(gpu, ora, [wl.beta_K], 0, sweep_slots=4096)
    n, _ = gpu.counts()
    assert n.max() > 1000 and (n > 0).mean() < 0.3  # U/R ~ 0.22, max n ~ 1e4


# ---------------------------------------------------------------------------------------------------
# parity reach (round 2): low temperatures at L = 128, zero temperature, theta = 1 at full size, u == T
# ---------------------------------------------------------------------------------------------------
def adopt(gpu, ora):
    """put the oracle into the GPU's state after a stretch of pa_run (population, beta, step ordinal, ln Z accumulator);
    E, M are recomputed by the oracle's own energy function and compared"""
    got = gpu.spins()
    E, M = gpu.energies()
    Eo, Mo = orc.energy_mag(ora.L, got)
    assert np.array_equal(E, Eo) and np.array_equal(M, Mo)
    ora.spins, ora.E, ora.M, ora.R = got, Eo, Mo, got.shape[0]
    ora.beta, ora.step_no = gpu.beta_steps()
    ora.sum_lnQ = gpu.log_Z()["sum_lnQ"]
    ora.part_start = orc.partition_table(ora.R, ora.P)


def test_L128_lockstep_down_to_beta_0p6():
    """config 4 shape at reduced R: 30 steps of dbeta = 0.02 (|dbeta| 2N = 655 < 700) reach beta = 0.6, the end of config
    4's schedule -- L = 128 sweeps compared on the whole population in the ordered phase, where almost every site
    needs a uniform and most of them are rejected"""
    gpu, ora = make_pair(128, 600, 148, seed=404)
    lockstep(gpu, ora, [0.02 * k for k in range(1, 31)], 2)
    assert gpu.observables()["mean_E"] / 128 ** 2 < -1.2  # a fast quench: domains, but deep in the low-energy region


def test_config4_full_size_sampled_late_in_the_schedule():
    """config 4 at full size, brought to beta = 0.45 and then to beta = 0.5988 by pa_run (its own schedule), with a
    lock-step step (a1-a6 on the whole population, theta = 20 sweeps on sampled slots) taken at each point"""
    wl = inputs.CONFIGS[4]
    gpu, ora = make_pair(wl.L, wl.R0, wl.P, wl.seed)
    k1, k2 = 375, 499
    assert gpu.run([wl.beta(k) for k in range(1, k1 + 1)], wl.theta) == k1
    adopt(gpu, ora)
    lockstep(gpu, ora, [wl.beta(k1 + 1)], wl.theta, sweep_slots=512)
    assert gpu.run([wl.beta(k) for k in range(k1 + 2, k2 + 1)], wl.theta) == k2 - k1 - 1
    adopt(gpu, ora)
    lockstep(gpu, ora, [wl.beta(k2 + 1)], wl.theta, sweep_slots=512)
    assert abs(gpu.beta_steps()[0] - 0.6) < 1e-12 and gpu.beta_steps()[1] == 500


@pytest.mark.parametrize("L", [8, 16, 64])
def test_zero_temperature_dynamics(L):
    """beta large enough that T4 = T8 = 0: deterministic zero-temperature dynamics (flip iff a >= 2), the regime the
    oracle's sweep is pinned in by hand (tests/test_oracle_pins.py::test_zero_temperature_dynamics_by_hand)"""
    R = 400
    pop = inputs.structured_population(L, R, seed=3 * L)
    step = 600.0 / (2 * L * L)  # |dbeta| 2N < 700 (reading G11)
    beta0 = 30.0
    gpu, ora = make_pair(L, R, P=3, seed=17, beta0=beta0, spins=pop, capacity=8 * R)
    lockstep(gpu, ora, [beta0 + step * k for k in range(1, 4)], 2)
    assert gpu.thresholds() == (0, 0)


def test_config3_full_size_theta1():
    """theta = 1 is the paper's scalability regime; full size, sampled slots"""
    wl = inputs.CONFIGS[3]
    gpu, ora = make_pair(wl.L, wl.R0, wl.P, wl.seed)
    lockstep(gpu, ora, [0.08, 0.16, 0.165], 1, sweep_slots=4096)


@pytest.mark.parametrize("L", [8, 32, 64])
def test_threshold_equal_to_the_uniform_is_not_accepted(L):
    """u == T (probability 2^-32 per site, never met by a temperature-derived threshold in any other test): with the
    test hook pa_debug_set_thresholds the thresholds are set to the very 32-bit uniform of one chosen site of an
    all-up lattice (every colour-0 site has a = 0 and compares against T8).  u < T is strict (C4): the site
    must stay; with T + 1 it must flip.  All 32 comparator bits are equal for that site, which takes the kernel to
    its last Philox block (c = 7)."""
    b = _binding()
    seed, R = 0x5EED0000 + L, 40
    half = L // 2
    y, k = L // 2 + 1, half - 1       # a site in the last group of its row block, colour 0
    q = y * half + k
    x = 2 * k + (y & 1)
    up = np.stack([orc.pack(L, np.ones(L * L, np.int8))] * R)
    for slot in (0, 2):
        for plus in (0, 1):
            g = b.PopulationAnnealer(L, R, seed=seed, capacity=256)
            g.set_spins(up)
            u = philox_ref.sweep_word(seed, 1, slot, 0, 0, q)  # step ordinal 1, sweep t = 0, colour 0
            T = min(u + plus, 0xFFFFFFFF)
            g.debug_set_thresholds(True, T4=0x12345678, T8=T)
            g.step(1e-9, 1)  # all energies are equal: tau = 1, R' ~ Poisson(40), every child is all-up again
            assert g.thresholds() == (0x12345678, T) and g.R > slot
            # oracle: the resampled population is all-up again (copies of identical parents); same thresholds
            want = np.stack([orc.pack(L, np.ones(L * L, np.int8))] * g.R)
            orc.sweeps(L, want, seed, 1, 1, 0x12345678, T)
            got = g.spins()
            assert np.array_equal(got, want)
            s = orc.unpack(L, got[slot]).reshape(L, L)
            # colour-0 site (x, y) was decided on the all-up lattice; colour 1 may have flipped neighbours afterwards but
            # never the site itself
            assert s[y, x] == (1 if plus == 0 else -1), (slot, plus)


def test_extreme_thresholds_through_the_hook():
    """T = 0 (never accept an uphill move) and T = 2^32 - 1 (accept unless u = 2^32 - 1) against the oracle"""
    b = _binding()
    L, R, seed = 32, 500, 99
    pop = inputs.random_packed_population(L, R, seed=5)
    for T4, T8 in [(0, 0), (0xFFFFFFFF, 0xFFFFFFFF), (0xFFFFFFFF, 0), (0x80000000, 0x7FFFFFFF)]:
        g = b.PopulationAnnealer(L, R, seed=seed, capacity=4096, flags=b.PA_KEEP_TAU | b.PA_KEEP_COUNTS)
        g.set_spins(pop)
        g.debug_set_thresholds(True, T4, T8)
        g.step(0.05, 2)
        o = orc.OraclePA(L, R, seed=seed, capacity=4096, spins=pop)
        o.resample(0.05, tau_override=g.tau())
        orc.sweeps(L, o.spins, seed, 1, 2, T4, T8)
        assert g.R == o.R and np.array_equal(g.spins(), o.spins), (T4, T8)
        g.debug_set_thresholds(False)
        g.step(0.1, 1)
        assert g.thresholds() == orc.thresholds(0.1)


@pytest.mark.parametrize("L", [8, 16, 32, 64, 128])
def test_every_threshold_bit_pair_in_every_position(L):
    """The sweep kernels of L >= 64 specialise the comparator on the pair (bit of T4, bit of T8) of each of the first 8
    bit positions -- four code paths per position, the first position with its own LUTs -- and the generic comparator
    takes over from bit 8 on.  Temperature-derived thresholds never produce T8 > T4 and reach few of the 4^8 patterns;
    the test hook sets crafted pairs that put every one of the four cases into every position (also T8 > T4: each class
    is compared with its own threshold, whatever their order), on a population with all neighbour classes."""
    b = _binding()
    R, seed, theta = (300 if L <= 32 else 64), 4242 + L, 2
    pop = inputs.random_packed_population(L, R, seed=L, p_up=0.75)  # plenty of sites with a = 0 and a = 1
    pairs = [(0x33333333, 0x55555555), (0x66666666, 0xAAAAAAAA), (0xCCCCCCCC, 0x55555555), (0x99999999, 0xAAAAAAAA),
             (0x0F0F3C3C, 0x3355CCAA), (0xF0F0C3C3, 0xCCAA3355)]  # the first four: case (p + i) mod 4 at position i
    seen = [set() for _ in range(8)]
    for T4, T8 in pairs:
        for i in range(8):
            seen[i].add((((T4 >> (31 - i)) & 1), ((T8 >> (31 - i)) & 1)))
        g = b.PopulationAnnealer(L, R, seed=seed, capacity=2048, flags=b.PA_KEEP_TAU | b.PA_KEEP_COUNTS)
        g.set_spins(pop)
        g.debug_set_thresholds(True, T4, T8)
        dbeta = min(0.02, 300.0 / (2 * L * L))
        g.step(dbeta, theta)
        assert g.thresholds() == (T4, T8)
        o = orc.OraclePA(L, R, seed=seed, capacity=2048, spins=pop)
        o.resample(dbeta, tau_override=g.tau())
        orc.sweeps(L, o.spins, seed, 1, theta, T4, T8)
        assert g.R == o.R and np.array_equal(g.spins(), o.spins), (hex(T4), hex(T8))
    assert all(len(sx) == 4 for sx in seen)


@pytest.mark.parametrize("L,R0", [(8, 620000), (16, 160000), (32, 40000)])
def test_wide_small_lattice_kernel_on_large_populations(L, R0):
    """k_sweep_small switches to 8 replicas per lane group once a population fills the GPU (L = 32: R0 >= 37 888, L = 16:
    151 552, L = 8: 606 208): full-population lock-step at those sizes, ferromagnet and a +-J sample"""
    for bonds in (None, inputs.bond_sample(L, 3 * L)):
        gpu, ora = make_pair(L, R0, 5, seed=77 + L, bonds=bonds)
        lockstep(gpu, ora, [0.1, 0.3, 0.45], theta=2)


@pytest.mark.parametrize("L,R0", [(8, 900), (32, 500), (64, 120)])
def test_heating_protocol_lockstep(L, R0):
    """PAPER.md:68 "the heating of the population": a population of ground states declared at a low temperature is
    annealed towards beta = 0 (negative dbeta, reading G29): lock-step with the oracle, every step"""
    N = L * L
    up = orc.pack(L, np.ones(N, np.int8))
    down = orc.pack(L, -np.ones(N, np.int8))
    spins = np.stack([up if j % 2 == 0 else down for j in range(R0)])
    beta0 = 1.0
    gpu, ora = make_pair(L, R0, 4, seed=31 + L, beta0=beta0, spins=spins)
    dbeta = min(0.08, 300.0 / (2 * N))
    betas = [beta0 - dbeta * k for k in range(1, 11)]
    lockstep(gpu, ora, betas, theta=2)
    assert gpu.log_Z()["sum_lnQ"] < 0.0 and rel(gpu.log_Z()["sum_lnQ"], ora.sum_lnQ) <= RTOL


@pytest.mark.parametrize("L,R0,theta", [(8, 1, 1), (8, 2049, 2), (16, 5000, 1), (32, 4097, 0), (64, 700, 2), (128, 90, 1),
                                        (8, 3000001, 0)])  # the last: 1465 tiles, more than one pass of the tile-prefix block
def test_systematic_resampling_lockstep(L, R0, theta):
    """A4c (PA_RESAMPLE_SYSTEMATIC): counts from the exact 64-bit cumulative weights on the device == the oracle's
    sequential loop, the population stays at R0 (+-1), lock-step over tile boundaries (2048 parents) and ragged sizes"""
    gpu, ora = make_pair(L, R0, 3, seed=900 + L, rule=2)
    dbeta = min(0.06, 300.0 / (2 * L * L))
    lockstep(gpu, ora, [dbeta * k for k in range(1, 7 if R0 < 100000 else 3)], theta=theta)
    assert abs(gpu.R - R0) <= 1


def test_systematic_resampling_on_a_skewed_population_and_without_the_keep_flags():
    b = _binding()
    L, R0 = 32, 20000
    spins = inputs.structured_population(L, R0, 5)
    gpu, ora = make_pair(L, R0, 148, seed=4, spins=spins, rule=2)   # copy counts of thousands per parent
    lockstep(gpu, ora, [0.03, 0.06], theta=0)
    lockstep(gpu, ora, [0.09], theta=1)
    assert abs(gpu.R - R0) <= 1
    # the timed configuration: no KEEP flags (the counts still travel through the n array), whole schedule in one call
    plain = b.PopulationAnnealer(L, R0, P=148, seed=4, flags=b.PA_RESAMPLE_SYSTEMATIC)
    plain.set_spins(spins)
    plain.run([0.03, 0.06], 0)
    plain.run([0.09], 1)
    assert plain.R == gpu.R and np.array_equal(plain.spins(), gpu.spins())
    with pytest.raises(b.PaError) as e:
        b.PopulationAnnealer(L, 100, flags=b.PA_RESAMPLE_SYSTEMATIC | b.PA_RESAMPLE_NEAREST)
    assert e.value.code == b.PA_EINVAL
    with pytest.raises(b.PaError) as e:
        b.PopulationAnnealer(L, 100, flags=b.PA_RESAMPLE_SYSTEMATIC, rank=0, world=2)
    assert e.value.code == b.PA_EINVAL


def test_failed_step_does_not_leak_into_the_getters():
    """after PA_ECAPACITY the getters of the last step refuse (their arrays hold the failed attempt) and last_Q is still
    the Q of the last committed step"""
    b = _binding()
    g = b.PopulationAnnealer(16, 1024, P=2, seed=3, capacity=1024, flags=b.PA_KEEP_TAU | b.PA_KEEP_COUNTS)
    k, failed = 0, False
    while not failed and k < 60:
        k += 1
        lz = g.log_Z()
        try:
            g.step(0.002 * k, 1)
        except b.PaError as e:
            assert e.code == b.PA_ECAPACITY
            failed = True
    assert failed
    assert g.log_Z() == lz
    for call in (g.tau, g.counts):
        with pytest.raises(b.PaError) as ei:
            call()
        assert ei.value.code == b.PA_EINVAL
    while True:  # the next committed step makes them valid again
        k += 1
        try:
            g.step(0.002 * k, 1)
            break
        except b.PaError:
            pass
    n, off = g.counts()
    assert int(n.sum()) == g.R == int(off[-1])


# ---------------------------------------------------------------------------------------------------
# variants of the step: nearest-integer resampling, adaptive temperature step
# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("L,R0,P,theta", [(8, 3000, 1, 2), (32, 4099, 7, 1), (64, 2048, 148, 2)])
def test_nearest_integer_resampling_lockstep(L, R0, P, theta):
    gpu, ora = make_pair(L, R0, P, seed=61 + L, rule=1)
    lockstep(gpu, ora, [0.07 * k for k in range(1, 8)], theta)
    assert abs(gpu.R - R0) < 5 * math.sqrt(R0 / 4)  # the population size barely moves under this rule


def test_nearest_integer_resampling_heavy_parents():
    # skewed weights: lambda up to hundreds -- the rule has no chunk loop, one uniform per parent whatever lambda is
    L, R = 32, 20000
    pop = inputs.random_packed_population(L, R, seed=5)
    pop[np.random.default_rng(7).choice(R, 64, replace=False)] = inputs.structured_population(L, 64, seed=6)
    gpu, ora = make_pair(L, R, P=3, seed=55, beta0=0.3, spins=pop, capacity=40960, rule=1)
    lockstep(gpu, ora, [0.304, 0.31], 1)
    assert gpu.counts()[0].max() > 8


@pytest.mark.parametrize("L,R0", [(16, 4000), (64, 3000)])
def test_adaptive_temperature_step(L, R0):
    """pa_adaptive_beta against the oracle's bisection on the same population, then a lock-step step to that temperature;
    the steps must shrink in the critical region"""
    gpu, ora = make_pair(L, R0, 5, seed=23)
    dbeta_max = min(0.05, 600.0 / (2 * L * L))
    steps = []
    while gpu.beta_steps()[0] < 0.46 and len(steps) < 250:  # past beta_c = 0.4407
        b_gpu = gpu.adaptive_beta(0.85, dbeta_max)
        b_ora = ora.adaptive_beta(0.85, dbeta_max)
        assert rel(b_gpu - ora.beta, b_ora - ora.beta) <= 1e-9, (b_gpu, b_ora)  # the bisection grids coincide unless a tie
        steps.append(b_gpu - ora.beta)
        lockstep(gpu, ora, [b_gpu], 1)
    assert gpu.beta_steps()[0] >= 0.46 and min(steps) < 0.7 * max(steps)
    with pytest.raises(_binding().PaError):
        gpu.adaptive_beta(1.5, 0.01)


# ---------------------------------------------------------------------------------------------------
# redistribution policies: partition tables, born / excess / shortage, moved
# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("policy,P,block,maxexc", [(1, 8, 1024, 1), (1, 8, 1024, 2), (1, 148, 64, 1), (1, 5, 1, 1),
                                                   (2, 8, 1024, 1), (2, 148, 1024, 1), (3, 8, 1024, 1), (3, 37, 1024, 1)])
def test_policies_lockstep(policy, P, block, maxexc):
    """lockstep() compares part_start, cnt/born/maxg/minl and `moved` with the oracle every step; the populations of the
    partitions drift apart under `none` and `naive`, which is what the paper's Fig. 1 shows"""
    gpu, ora = make_pair(64, 8 * 2048 + 77, P, seed=31 + policy, policy=policy, block=block, maxexc=maxexc)
    lockstep(gpu, ora, [0.06 * k for k in range(1, 9)], 1)   # up to beta = 0.48, across beta_c
    ps, st, moved = gpu.partitions()
    if policy == 3:
        assert moved == 0 and np.array_equal(st[:, 0], st[:, 1])
        assert st[:, 0].max() > 1.2 * st[:, 0].mean()  # partitions have drifted apart
    if policy == 1:
        r = np.diff(orc.partition_table(gpu.R, P).astype(np.int64))
        assert np.all(np.abs(st[:, 0].astype(np.int64) - r) <= maxexc * block)


def test_policy_arguments_are_validated():
    b = _binding()
    with pytest.raises(b.PaError):
        b.PopulationAnnealer(8, 64, P=4, policy=7)
    with pytest.raises(b.PaError):
        b.PopulationAnnealer(8, 5000, P=2000, policy=b.PA_POLICY_MAIN)  # P <= 1024 for the paper's policies
    b.PopulationAnnealer(8, 5000, P=2000)  # the balanced table has no such limit


# ---------------------------------------------------------------------------------------------------
# multi-GPU partitioned redistribution: the ranks of a sharded run, emulated on ONE device and stepped
# phase by phase by the host, must reproduce the single-context run bit for bit
# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("world,L,R0,theta,policy", [(2, 32, 5000, 2, 0), (4, 64, 3001, 1, 0), (3, 16, 4099, 0, 0),
                                                     (2, 64, 2500, 3, 1), (3, 32, 3000, 1, 2), (2, 8, 4000, 2, 3),
                                                     (5, 128, 700, 1, 0)])
def test_sharded_ranks_equal_the_single_context(world, L, R0, theta, policy):
    b = _binding()
    from paper_2006_00561_b200 import dist
    seed = 1000 + 7 * world + L
    single = b.PopulationAnnealer(L, R0, P=1, seed=seed)
    sh = dist.ShardedAnnealer(L, R0, seed=seed, policy=policy, block=64, maxexc=1, emulate=world)
    assert np.array_equal(sh.gather_spins(), single.spins())  # the initial population is keyed by global replica index
    dbeta = min(0.05, 600.0 / (2 * L * L))
    for k in range(1, 7):
        single.step(dbeta * k, theta)
        obs = sh.step(dbeta * k, theta)
        assert sum(sh.R_local) == single.R == sum(o["R"] for o in obs)
        assert np.array_equal(sh.gather_spins(), single.spins()), (k, "spins")
        so = single.observables()
        for key in ["sum_E", "sum_E2", "sum_absM", "sum_M2", "sum_M4"]:
            assert sum(o[key] for o in obs) == so[key], (k, key)
        for s_ in sh.shards:  # every rank carries the same ln Z (the ranks' weight sums are added in rank order)
            assert rel(s_.log_Z()["lnZ"], single.log_Z()["lnZ"]) <= RTOL
        E = np.concatenate([s_.energies()[0] for s_ in sh.shards])
        assert np.array_equal(E, single.energies()[0])
        # what the plan moved is what the ranks hold
        ns = sh.last_new_start
        assert [int(ns[r + 1] - ns[r]) for r in range(world)] == sh.R_local
        if policy == 3:
            assert np.array_equal(np.asarray(sh.last_counts), np.diag(sh.last_T))


def test_sharded_driver_with_one_rank_equals_the_single_context():
    """the non-emulated driver path (the one torchrun ranks take), world size 1"""
    b = _binding()
    from paper_2006_00561_b200 import dist
    single = b.PopulationAnnealer(32, 3000, seed=4)
    sh = dist.ShardedAnnealer(32, 3000, seed=4, group=dist.Group())
    for k in range(1, 5):
        single.step(0.1 * k, 2)
        sh.step(0.1 * k, 2)
        assert np.array_equal(sh.gather_spins(), single.spins())
        assert rel(sh.log_Z()["lnZ"], single.log_Z()["lnZ"]) <= RTOL  # Q's rounding depends on the reduction grid (capacity)


def _two_process_rank(rank, world, port, q, L, R0, seed, betas, theta, policy):
    """one REAL rank of the multi-process driver: its own process, its own CUDA context on cuda:0, torch.distributed over
    gloo with host-staged slices.  Kernels of different ranks never wait on one another (the ranks meet on the host)."""
    os.environ.update({"RANK": str(rank), "WORLD_SIZE": str(world), "LOCAL_RANK": "0",
                       "MASTER_ADDR": "127.0.0.1", "MASTER_PORT": str(port)})
    import torch
    from paper_2006_00561_b200 import dist
    g = dist.init_from_env(backend="gloo", device_kind="cuda")
    sh = dist.ShardedAnnealer(L, R0, seed=seed, policy=policy, block=64, maxexc=1, group=g)
    Rs = []
    for beta in betas:
        sh.step(beta, theta)
        Rs.append(sh.R_local[0])
    torch.cuda.synchronize()
    q.put((rank, sh.shards[0].spins(), sh.shards[0].energies()[0], sh.log_Z()["lnZ"], Rs, int(sh.last_new_start[rank])))
    dist.barrier(g)
    dist.shutdown(g)


@pytest.mark.parametrize("world,policy", [(2, 0), (3, 1)])
def test_sharded_real_processes_on_one_gpu_equal_the_single_context(world, policy):
    """the multi-process driver path (dist.init_from_env, all_gather_doubles, exchange_slices, ShardedAnnealer(group=...))
    executed with world > 1: `world` spawned processes share cuda:0, exchange over gloo; the concatenation of their
    populations equals the single-context run bit for bit, step counts and ln Z agree on every rank"""
    import socket
    import torch.multiprocessing as mp
    b = _binding()
    L, R0, seed, theta = 32, 3000, 31, 2
    betas = [0.08 * k for k in range(1, 7)]
    s_ = socket.socket()
    s_.bind(("127.0.0.1", 0))
    port = s_.getsockname()[1]
    s_.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_two_process_rank, args=(r, world, port, q, L, R0, seed, betas, theta, policy)) for r in range(world)]
    for p_ in procs:
        p_.start()
    res = sorted((q.get(timeout=300) for _ in procs), key=lambda t: t[0])
    for p_ in procs:
        p_.join(timeout=120)
        assert p_.exitcode == 0
    single = b.PopulationAnnealer(L, R0, P=1, seed=seed)
    Rs = []
    for beta in betas:
        single.step(beta, theta)
        Rs.append(single.R)
    assert np.array_equal(np.concatenate([r[1] for r in res], axis=0), single.spins())
    assert np.array_equal(np.concatenate([r[2] for r in res]), single.energies()[0])
    assert [sum(r[4][k] for r in res) for k in range(len(betas))] == Rs
    starts = [r[5] for r in res]
    assert starts[0] == 0 and starts == sorted(starts)
    for r in res:
        assert rel(r[3], single.log_Z()["lnZ"]) <= RTOL


def test_sharded_capacity_failure_is_consistent_and_leaves_the_population_unchanged():
    b = _binding()
    from paper_2006_00561_b200 import dist
    sh = dist.ShardedAnnealer(16, 2048, seed=5, capacity=1100, emulate=2)  # 1024 per rank, almost no slack
    failures = 0
    for k in range(1, 40):
        before, Rb, lz = sh.gather_spins(), sh.R_local, sh.log_Z()
        try:
            sh.step(0.003 * k, 1)
        except b.PaError as e:
            assert e.code == b.PA_ECAPACITY
            failures += 1
            assert sh.R_local == Rb and np.array_equal(sh.gather_spins(), before) and sh.log_Z() == lz
    assert failures > 0


def test_sharded_empty_share_is_refused_by_all_ranks_before_the_exchange():
    """policy none and one replica or two per rank: sooner or later a rank has no offspring.  A shard cannot be empty, and
    the refusal must come from the plan check on EVERY rank (same gathered totals) before anything is exchanged or
    committed -- not from the one empty rank's pa_dist_finish after the others have committed"""
    b = _binding()
    from paper_2006_00561_b200 import dist
    sh = dist.ShardedAnnealer(8, 6, seed=3, policy=b.PA_POLICY_NONE, emulate=2, flags=b.PA_KEEP_COUNTS)
    refused = committed = 0
    for k in range(1, 400):  # (a refused step keeps its ordinal, hence its random numbers: the retries mostly fail again)
        if refused >= 3:
            break
        before, Rb, lz, bs = sh.gather_spins(), sh.R_local, sh.log_Z(), [s_.beta_steps() for s_ in sh.shards]
        try:
            sh.step(0.002 * k, 1)
            committed += 1
            assert len(set(s_.beta_steps() for s_ in sh.shards)) == 1           # same beta and step ordinal on all ranks
        except b.PaError as e:
            assert e.code in (b.PA_EEXTINCT, b.PA_ECAPACITY)
            refused += 1
            assert sh.R_local == Rb and np.array_equal(sh.gather_spins(), before) and sh.log_Z() == lz
            assert [s_.beta_steps() for s_ in sh.shards] == bs
            for s_ in sh.shards:                                                 # the dropped attempt's arrays are not served
                with pytest.raises(b.PaError):
                    s_.counts()
    assert refused > 0 and committed > 0


# ---------------------------------------------------------------------------------------------------
# boundary behaviour
# ---------------------------------------------------------------------------------------------------
def test_run_equals_repeated_step_and_is_deterministic():
    b = _binding()
    betas = [0.05 * k for k in range(1, 9)]
    a = b.PopulationAnnealer(32, 3000, P=4, seed=9)
    for beta in betas:
        a.step(beta, 2)
    c = b.PopulationAnnealer(32, 3000, P=4, seed=9)
    assert c.run(betas, 2) == len(betas)
    assert a.R == c.R and np.array_equal(a.spins(), c.spins())
    assert a.log_Z() == c.log_Z() and a.observables() == c.observables()
    assert a.beta_steps() == c.beta_steps() == (betas[-1], len(betas))


def test_run_longer_than_the_parameter_ring():
    """pa_run uploads step parameters in chunks of 1024: a schedule of 2100 steps in one call equals the same schedule
    in three calls (and the oracle at a few check points would be slow: determinism + ln Z continuity is the check)"""
    b = _binding()
    betas = [2e-4 * k for k in range(1, 2101)]
    a = b.PopulationAnnealer(8, 300, P=3, seed=12)
    assert a.run(betas, 1) == 2100
    c = b.PopulationAnnealer(8, 300, P=3, seed=12)
    assert c.run(betas[:7], 1) + c.run(betas[7:1500], 1) + c.run(betas[1500:], 1) == 2100
    assert a.R == c.R and np.array_equal(a.spins(), c.spins())
    assert a.log_Z() == c.log_Z() and a.observables() == c.observables() and a.beta_steps() == c.beta_steps()
    ora = orc.OraclePA(8, 300, P=3, seed=12)
    for beta in betas[:40]:
        ora.step(beta, 1)
    d = b.PopulationAnnealer(8, 300, P=3, seed=12)
    d.run(betas[:40], 1)
    compare_population(d, ora, "40 steps")  # counts come from each side's own tau here: equal unless a 1e-16 tie


def test_capacity_error_leaves_population_unchanged():
    b = _binding()
    g = b.PopulationAnnealer(16, 1024, P=2, seed=3, capacity=1024)
    failures = 0
    for k in range(1, 60):
        before, R_before, lz_before, bs = g.spins(), g.R, g.log_Z(), g.beta_steps()
        try:
            g.step(0.002 * k, 1)
        except b.PaError as e:
            assert e.code == b.PA_ECAPACITY
            failures += 1
            assert g.R == R_before and np.array_equal(g.spins(), before)
            assert g.log_Z() == lz_before and g.beta_steps() == bs
    assert failures > 5  # R' ~ Poisson(1024) exceeds 1024 about half of the time
    assert g.beta_steps()[1] == 59 - failures


def test_extinction_matches_the_oracle_and_leaves_population_unchanged():
    """degenerate case R' = 0 (PA_EEXTINCT): R0 = 2 replicas die out with probability e^-2 per step; the first seed on
    which the ORACLE goes extinct must make the GPU fail at the same step, with nothing committed"""
    b = _binding()
    hit = None
    for seed in range(40):
        ora = orc.OraclePA(8, 2, seed=seed)
        try:
            for k in range(1, 6):
                ora.step(0.01 * k, 1)
        except orc.OracleError:
            hit = (seed, k)
            break
    assert hit is not None
    seed, kfail = hit
    g = b.PopulationAnnealer(8, 2, seed=seed)
    for k in range(1, kfail):
        g.step(0.01 * k, 1)
    before, R_before, lz, bs = g.spins(), g.R, g.log_Z(), g.beta_steps()
    with pytest.raises(b.PaError) as ei:
        g.step(0.01 * kfail, 1)
    assert ei.value.code == b.PA_EEXTINCT
    assert g.R == R_before and np.array_equal(g.spins(), before) and g.log_Z() == lz and g.beta_steps() == bs
    assert np.array_equal(before, ora.spins) and R_before == ora.R  # oracle state is also the pre-step one


def test_invalid_arguments():
    b = _binding()
    with pytest.raises(b.PaError):
        b.PopulationAnnealer(12, 100)  # unsupported L
    with pytest.raises(b.PaError):
        b.PopulationAnnealer(8, 0)
    g = b.PopulationAnnealer(8, 64)
    for bad in [lambda: g.step(float("nan"), 1), lambda: g.step(0.1, -1), lambda: g.step(-0.1, 1),
                lambda: g.step(1e4, 0), lambda: g.spins(0, 65), lambda: g.tau()]:
        with pytest.raises(b.PaError) as ei:
            bad()
        assert ei.value.code == b.PA_EINVAL
    g.step(0.1, 1)  # still usable


def test_global_flip_covariance_on_gpu():
    b = _binding()
    pop = inputs.random_packed_population(64, 500, seed=8)
    a = b.PopulationAnnealer(64, 500, seed=77)
    c = b.PopulationAnnealer(64, 500, seed=77)
    a.set_spins(pop)
    c.set_spins(~pop)
    for k in range(1, 7):
        a.step(0.08 * k, 3)
        c.step(0.08 * k, 3)
        assert np.array_equal(a.spins(), ~c.spins())
        Ea, Ma = a.energies()
        Ec, Mc = c.energies()
        assert np.array_equal(Ea, Ec) and np.array_equal(Ma, -Mc)
        assert a.log_Z() == c.log_Z()


def test_device_getters_and_launch_count():
    b = _binding()
    g = b.PopulationAnnealer(32, 2000, seed=4, flags=b.PA_PROFILE)
    g.profile_read()  # drain the launches of pa_init
    l0 = g.launch_count()
    g.step(0.1, 2)
    assert g.launch_count() - l0 == 4  # q_reduce (+ level tables), poisson_scan (+ child -> parent map), sweep (gathers), observe (+ a5)
    Ed, Md = g.energies_device()
    E, M = g.energies()
    assert np.array_equal(Ed.cpu().numpy(), E) and np.array_equal(Md.cpu().numpy(), M)
    prof = g.profile_read()
    assert all(cnt == (0 if k in ("balance", "levels_w", "levels_tau", "copy") else 1) for k, (_, cnt) in prof.items()) and prof["sweep"][0] > 0
    g.profile_read()
    l1 = g.launch_count()  # (the getters above launched their unpack kernels)
    g.step(0.2, 0)  # theta = 0: the gather copy runs instead of the sweep
    prof = g.profile_read()
    assert prof["copy"][1] == 1 and prof["sweep"][1] == 0 and g.launch_count() - l1 == 4


def test_bench_line_carries_the_contract_keys():
    """bench.py (our arm, config 1 to keep it short): one JSON line with the driver contract's keys, the roofline /
    e2e / cpu_baseline objects of the tier framing, and a non-zero count of OUR kernel launches"""
    import json
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    out = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--config", "1", "--steps", "5", "--warmup", "3",
                          "--no-resample"], capture_output=True, text=True, timeout=600, check=True).stdout
    line = json.loads(out.strip().splitlines()[-1])
    for key in ["metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
                "vs_baseline", "dtype", "data", "config", "clocks", "e2e", "gpu_launches", "roofline", "cpu_baseline"]:
        assert key in line, key
    assert line["metric"] == "spin_flip_attempts_per_s" and line["steps"] == 5 and line["n_gpus"] == 1
    assert line["value"] > 0 and line["gpu_launches"] == 5 * 4 and line["data"] == "synthetic"
    assert line["config"]["workload"].startswith("config1") and line["vs_baseline"] is None
    assert set(["bound", "achieved", "peak", "unit", "frac", "traffic"]) <= set(line["roofline"])
    assert line["e2e"]["h2d_bytes_per_step"] > 0 and line["e2e"]["d2h_bytes_per_step"] > 0 and line["e2e"]["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] >= 1
