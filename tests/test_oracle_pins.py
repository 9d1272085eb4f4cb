"""Pins for the CPU oracle (-m "not gpu"): every routine of oracle/pa_oracle.c is checked against something
other than itself -- closed forms, brute force, exact finite-lattice results, statistical laws, or an
independent big-integer writing of Philox.  Citations: PAPER.md line + equation; reading ids."""
import json
import math
import os

import numpy as np
import pytest
from mpmath import mp, mpf
from scipy import stats

from oracle import pa_oracle as orc

import exact_ising
import philox_ref

GOLD = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "ising_exact.json")))


# ---------------------------------------------------------------------------------------------------
# exact results themselves (pin the pins): Kaufman vs brute force, vs Onsager, vs beta->0 moments
# ---------------------------------------------------------------------------------------------------
def test_kaufman_matches_bruteforce_L4_and_golden():
    dos, _ = exact_ising.brute_force_dos(4)
    assert {str(k): v for k, v in dos.items()} == GOLD["dos_L4"]
    assert sum(dos.values()) == 65536
    for b in [0.005, 0.1, 0.4407, 0.5, 0.6, 1.0]:
        k = exact_ising.kaufman_lnZ(4, b)
        d = exact_ising.lnZ_from_dos(dos, b)
        assert abs(k - d) < mpf(10) ** -40
        assert abs(k - mpf(GOLD["lnZ"]["L4_beta%g" % b])) < mpf(10) ** -25


def test_kaufman_golden_values_and_survey_quotes():
    # SURVEY.md 8(c) "Reference values (survey check, mpmath 60 digits)"
    survey = {(8, 1.0): 128.715437337408418, (8, 0.5): 66.344581879227808, (16, 1.0): 512.78230780794178,
              (32, 1.0): 2049.0497896900873, (64, 0.5): 4202.3405079789426, (128, 0.6): 19827.502196897917}
    for (L, b), v in survey.items():
        k = exact_ising.kaufman_lnZ(L, b)
        assert abs(float(k) - v) <= 1e-13 * abs(v)
        assert abs(k - mpf(GOLD["lnZ"]["L%d_beta%g" % (L, b)])) < mpf(10) ** -22


def test_kaufman_high_temperature_moments_and_onsager_limit():
    # at beta=0: lnZ = N ln2, d lnZ/d beta = -<E> = 0, d2 lnZ/d beta2 = Var(E) = number of bonds = 2N
    mp.dps = 60
    L, N, h = 8, 64, mpf("1e-8")
    f = lambda b: exact_ising.kaufman_lnZ(L, b)
    f0 = N * mp.log(2)
    d1 = (f(h) - f0) / h
    d2 = (f(2 * h) - 2 * f(h) + f0) / h ** 2
    assert abs(d1) < 1e-5
    assert abs(d2 - 2 * N) < 1e-3
    # ordered phase: lnZ_L - N * onsager -> ln 2 (two ground states), SURVEY.md 8(c) "Onsager limit"
    for L, b in [(64, 0.6), (128, 0.6), (32, 1.0)]:
        diff = exact_ising.kaufman_lnZ(L, b) - L * L * exact_ising.onsager_lnZ_per_site(b)
        assert abs(diff - mp.log(2)) < 1e-6


# ---------------------------------------------------------------------------------------------------
# C3 Philox
# ---------------------------------------------------------------------------------------------------
def test_philox_against_bigint_writing():
    rng = np.random.default_rng(123)
    cases = [([0, 0, 0, 0], [0, 0]), ([0xFFFFFFFF] * 4, [0xFFFFFFFF] * 2), ([1, 2, 3, 4], [5, 6])]
    for _ in range(2000):
        cases.append((rng.integers(0, 2 ** 32, 4, dtype=np.uint64).tolist(),
                      rng.integers(0, 2 ** 32, 2, dtype=np.uint64).tolist()))
    for ctr, key in cases:
        assert orc.philox4x32_10(ctr, key).tolist() == philox_ref.philox4x32_10(ctr, key)


def test_philox_output_looks_uniform():
    # bit balance over 4000 consecutive counters: a stuck/constant word fails this
    words = np.array([orc.philox4x32_10([i, 7, 0, 0], [42, 0]) for i in range(4000)], dtype=np.uint32)
    bits = np.unpackbits(words.view(np.uint8)).mean()
    assert abs(bits - 0.5) < 0.005
    assert len(np.unique(words)) == words.size


# ---------------------------------------------------------------------------------------------------
# C1 energy / magnetisation, C2 layout
# ---------------------------------------------------------------------------------------------------
def test_energy_bruteforce_L4_density_of_states_and_Z():
    L = 4
    states = np.arange(65536, dtype=np.uint32).reshape(-1, 1)  # N=16 bits: the packed word IS the state index
    E, M = orc.energy_mag(L, states)
    dos_ref, E_ref = exact_ising.brute_force_dos(L)
    assert np.array_equal(E, E_ref)  # independent numpy-roll energy, state by state
    vals, counts = np.unique(E, return_counts=True)
    assert {str(int(v)): int(c) for v, c in zip(vals, counts)} == GOLD["dos_L4"]
    pop = np.array([bin(i).count("1") for i in range(65536)])
    assert np.array_equal(M, 2 * pop - 16)
    for b in [0.1, 0.4407, 1.0]:  # PAPER.md:33 eq. 1 summed over all states with the ORACLE's energies
        Z = sum(mp.exp(-mpf(b) * int(e)) * int(c) for e, c in zip(vals, counts))
        assert abs(mp.log(Z) - exact_ising.kaufman_lnZ(L, b)) < 1e-25


@pytest.mark.parametrize("L", [4, 8, 16, 32, 64])
def test_energy_special_configurations(L):
    N = L * L
    up = np.ones(N, np.int8)
    assert orc.energy_int8(L, up) == -2 * N
    assert orc.energy_int8(L, -up) == -2 * N
    yy, xx = np.divmod(np.arange(N), L)
    checker = np.where((xx + yy) % 2 == 0, 1, -1).astype(np.int8)
    assert orc.energy_int8(L, checker) == 2 * N
    rows = np.where(yy % 2 == 0, 1, -1).astype(np.int8)  # horizontal bonds satisfied, vertical all broken
    cols = np.where(xx % 2 == 0, 1, -1).astype(np.int8)
    assert orc.energy_int8(L, rows) == 0 and orc.energy_int8(L, cols) == 0
    one = up.copy()
    one[5 * L + 3 if L > 5 else 1 * L + 2] = -1
    assert orc.energy_int8(L, one) == -2 * N + 8
    # a domain wall pair: rows 0..h-1 down, rest up -> 2L broken vertical bonds -> E = -2N + 4L
    wall = np.where(yy < L // 2, -1, 1).astype(np.int8)
    assert orc.energy_int8(L, wall) == -2 * N + 4 * L
    wallx = np.where(xx < L // 2, -1, 1).astype(np.int8)
    assert orc.energy_int8(L, wallx) == -2 * N + 4 * L


@pytest.mark.parametrize("L", [8, 32])
def test_energy_symmetries_and_layout(L):
    rng = np.random.default_rng(L)
    N = L * L
    s = rng.choice(np.array([-1, 1], np.int8), size=(50, N))
    packed = np.stack([orc.pack(L, r) for r in s])
    E, M = orc.energy_mag(L, packed)
    assert np.all(E % 4 == 0) and np.all(np.abs(E) <= 2 * N)
    E2, M2 = orc.energy_mag(L, ~packed)  # global flip: E(sigma) = E(-sigma), M -> -M
    assert np.array_equal(E, E2) and np.array_equal(M, -M2)
    assert np.array_equal(M, s.sum(axis=1))
    # C2: bit b = y*L + x of the little-endian bit string, bit 1 <-> +1
    for r, p in zip(s[:5], packed[:5]):
        bits = np.unpackbits(p.view(np.uint8), bitorder="little")[:N]
        assert np.array_equal(bits.astype(np.int8) * 2 - 1, r)
        assert np.array_equal(orc.unpack(L, p), r)
    # energy from numpy rolls (second writing of eq. 6)
    g = s.reshape(-1, L, L).astype(np.int64)
    Eref = -(g * np.roll(g, -1, 2)).sum((1, 2)) - (g * np.roll(g, -1, 1)).sum((1, 2))
    assert np.array_equal(E, Eref)


# ---------------------------------------------------------------------------------------------------
# A1 init
# ---------------------------------------------------------------------------------------------------
def test_init_population_keying_and_statistics():
    L, R, seed = 32, 2000, 0x1234567887654321
    pop = orc.init_population(L, R, seed)
    assert pop.shape == (R, 32)
    for j in [0, 1, 777, 1999]:
        for v in [0, 1, 5, 31]:
            assert int(pop[j, v]) == philox_ref.init_word(seed, j, v)
    E, M = orc.energy_mag(L, pop)
    N = L * L
    # uniform spins: <M>=0, Var M = N; <E>=0, Var E = 2N (2N independent +-1 bonds)
    assert abs(M.mean()) < 5 * math.sqrt(N / R)
    assert abs(M.var() / N - 1) < 0.15
    assert abs(E.mean()) < 5 * math.sqrt(2 * N / R)
    assert abs(E.var() / (2 * N) - 1) < 0.15


# ---------------------------------------------------------------------------------------------------
# C5: Q (eq. 3), tau (eq. 4)
# ---------------------------------------------------------------------------------------------------
def test_q_tau_closed_forms():
    R = 1000
    E = np.full(R, -40, np.int32)
    Q = orc.q_ratio(E, 0.01)
    assert abs(Q - math.exp(0.4)) <= 4e-16 * Q
    assert np.allclose(orc.tau_weights(E, 0.01, Q), 1.0, rtol=1e-15, atol=0)
    # two-level population: a copies at E1, b at E2
    a, b, E1, E2, db = 300, 700, -64, 16, 0.05
    E = np.array([E1] * a + [E2] * b, np.int32)
    Qref = (a * mp.exp(-mpf(db) * E1) + b * mp.exp(-mpf(db) * E2)) / (a + b)
    Q = orc.q_ratio(E, db)
    assert abs(Q - float(Qref)) <= 1e-15 * Q
    tau = orc.tau_weights(E, db, Q)
    assert abs(tau[0] - float(mp.exp(-mpf(db) * E1) / Qref)) <= 1e-15 * tau[0]
    assert abs(tau[-1] - float(mp.exp(-mpf(db) * E2) / Qref)) <= 1e-15 * tau[-1]
    # sign convention: lowering the temperature (dbeta>0) favours LOW energy
    assert tau[0] > 1 > tau[-1]


def test_q_normalised_by_current_population_and_sum_tau():
    rng = np.random.default_rng(7)
    N = 1024
    for R in [1, 17, 4096, 100003]:
        E = (4 * rng.integers(-N // 4, N // 4, R)).astype(np.int32)
        db = 0.005
        Q = orc.q_ratio(E, db)
        ref = mp.fsum([mp.exp(-mpf(db) * int(e)) for e in E[:5000]]) / min(R, 5000) if R <= 5000 else None
        if ref is not None:
            assert abs(Q - float(ref)) <= 1e-14 * Q
        tau = orc.tau_weights(E, db, Q)
        assert abs(math.fsum(tau) - R) <= 1e-12 * R  # sum_j tau_j = R  (eq. 3 + eq. 4)
        Ql = orc.q_ratio_by_levels(E, db, N)
        assert abs(Ql - Q) <= 1e-14 * Q


# ---------------------------------------------------------------------------------------------------
# A4 Poisson sampler
# ---------------------------------------------------------------------------------------------------
def test_expneg_accuracy():
    mp.dps = 40
    worst = 0.0
    for mu in list(np.linspace(0, 8, 2001)) + [1e-300, 1e-17, 7.999999999, 8.0]:
        got = orc.expneg(mu)
        ref = mp.exp(-mpf(float(mu)))
        ulp = math.ulp(float(ref))
        worst = max(worst, abs(mpf(got) - ref) / ulp)
    assert worst <= 32, worst  # DESIGN.md A4: <= 32 ulp on [0, 8]
    assert orc.expneg(0.0) == 1.0


def test_uniform_resample_exact_bits():
    seed, step = 0xDEADBEEFCAFEF00D, 17
    for j in [0, 3, 65535, 2 ** 24 - 1]:
        for c in [0, 1, 2, 3, 1249]:
            u = orc.uniform_resample(seed, step, j, c)
            num = philox_ref.resample_uniform_fraction(seed, step, j, c)
            assert 0.0 < u < 1.0
            assert u == num / 2.0 ** 53  # exact in binary64


def _counts(lam, n, seed=99, step=3):
    return orc.poisson_counts(np.full(n, lam), 1.0, seed, step).astype(np.int64)


@pytest.mark.parametrize("lam,n", [(0.01, 400000), (1.0, 400000), (7.99, 200000), (8.01, 200000), (100.0, 50000),
                                   (1.0e4, 1500)])
def test_poisson_mean_and_variance(lam, n):
    k = _counts(lam, n)
    se_mean = math.sqrt(lam / n)
    assert abs(k.mean() - lam) < 5 * se_mean
    # Var of sample variance for Poisson ~ (lam + 2 lam^2)/n
    se_var = math.sqrt((lam + 2 * lam * lam) / n)
    assert abs(k.var() - lam) < 5 * se_var


def test_poisson_chi_square_lambda_1_and_5():
    for lam in [1.0, 5.0]:
        n = 400000
        k = _counts(lam, n, seed=5)
        kmax = int(stats.poisson.ppf(1 - 1e-5, lam))
        obs = np.bincount(np.minimum(k, kmax), minlength=kmax + 1).astype(float)
        p = stats.poisson.pmf(np.arange(kmax + 1), lam)
        p[-1] = 1 - p[:-1].sum()
        chi2 = ((obs - n * p) ** 2 / (n * p)).sum()
        assert chi2 < stats.chi2.ppf(1 - 1e-6, kmax)


def test_poisson_is_cdf_inversion_of_the_keyed_uniform():
    # one chunk (lam <= 8): n = smallest k with u <= F(k); compare with scipy's ppf of the SAME u
    seed, step, lam = 31337, 9, 3.7
    js = np.arange(20000)
    n = np.array([orc.poisson(lam, seed, step, int(j)) for j in js])
    u = np.array([orc.uniform_resample(seed, step, int(j), 0) for j in js])
    ref = stats.poisson.ppf(u, lam).astype(np.int64)
    # boundaries agree except where u is within rounding of a CDF step (none expected in 2e4 draws)
    assert (n != ref).sum() <= 1
    # two chunks (8 < lam <= 16): sum of two inversions at mu = lam/2 with uniforms c=0,1
    lam = 11.0
    n2 = np.array([orc.poisson(lam, seed, step, int(j)) for j in js[:5000]])
    u0 = np.array([orc.uniform_resample(seed, step, int(j), 0) for j in js[:5000]])
    u1 = np.array([orc.uniform_resample(seed, step, int(j), 1) for j in js[:5000]])
    ref2 = (stats.poisson.ppf(u0, lam / 2) + stats.poisson.ppf(u1, lam / 2)).astype(np.int64)
    assert (n2 != ref2).sum() <= 1


def test_poisson_degenerate_inputs():
    assert orc.poisson(0.0, 1, 1, 0) == 0
    assert orc.poisson(-1.0, 1, 1, 0) == 0
    assert orc.poisson(float("nan"), 1, 1, 0) == 0
    assert orc.poisson(1e-300, 1, 1, 0) == 0
    # scale factor: lambda = tau * R0/R (reading G2)
    tau = np.full(100000, 1.0)
    n_half = orc.poisson_counts(tau, 0.5, 4, 1)
    assert abs(n_half.mean() - 0.5) < 5 * math.sqrt(0.5 / tau.size)


# ---------------------------------------------------------------------------------------------------
# A4b nearest-integer resampling, A9 adaptive temperature step (readings G24, G25)
# ---------------------------------------------------------------------------------------------------
def test_nearest_integer_resampling():
    seed, step = 4242, 6
    for lam in [0.0, 0.3, 1.0, 2.75, 17.5, 1234.001]:
        n = np.array([orc.nearest(lam, seed, step, j) for j in range(20000)])
        assert set(np.unique(n)) <= {math.floor(lam), math.floor(lam) + 1}   # one of the two neighbouring integers
        f = lam - math.floor(lam)
        assert abs(n.mean() - lam) <= 5 * math.sqrt(max(f * (1 - f), 1e-12) / n.size) + 1e-12   # E[n] = lambda
        if f == 0.0:
            assert np.all(n == int(lam))                                     # integer lambda: no randomness at all
    # the decision uses the keyed uniform of chunk 0 of parent j: n = floor + [u > 1 - frac]
    lam = 3.37
    for j in [0, 5, 999]:
        u = orc.uniform_resample(seed, step, j, 0)
        assert orc.nearest(lam, seed, step, j) == 3 + (1 if u > 1.0 - (lam - 3.0) else 0)
    assert orc.nearest(-1.0, 1, 1, 0) == 0 and orc.nearest(float("nan"), 1, 1, 0) == 0
    # population size: sum_j n_j stays within a few sqrt(R/4) of R0 (Poisson: sqrt(R0))
    rng = np.random.default_rng(1)
    tau = rng.gamma(2.0, 0.5, 50000)
    tau *= tau.size / tau.sum()
    tot = int(orc.nearest_counts(tau, 1.0, seed, step).sum())
    assert abs(tot - tau.size) < 5 * math.sqrt(tau.size / 4)
    pa = orc.OraclePA(8, 2000, seed=3, rule=orc.RULE_NEAREST)
    sizes = [pa.step(0.05 * k, 2)["Rnew"] for k in range(1, 11)]
    assert max(abs(s - 2000) for s in sizes) < 5 * math.sqrt(2000 / 4)
    assert abs(pa.lnZ - float(exact_ising.kaufman_lnZ(8, 0.5))) < 0.5         # still a valid PA estimate of ln Z


def test_overlap_closed_forms_and_adaptive_step():
    # all energies equal: every tau = 1 -> overlap 1 for any dbeta
    E = np.full(500, -24, np.int32)
    assert orc.overlap(E, 0.3) == 1.0
    # two levels: a replicas at E1, b at E2 (E1 < E2, dbeta > 0): tau1 > 1 > tau2 -> alpha = (a + b tau2) / (a + b)
    a, b, E1, E2, db = 300, 700, -64, 16, 0.02
    E = np.array([E1] * a + [E2] * b, np.int32)
    w1, w2 = mp.exp(-mpf(db) * E1), mp.exp(-mpf(db) * E2)
    Q = (a * w1 + b * w2) / (a + b)
    want = float((a + b * w2 / Q) / (a + b))
    assert abs(orc.overlap(E, db) - want) <= 1e-14
    rng = np.random.default_rng(12)
    E = (4 * rng.integers(-300, 300, 20000)).astype(np.int32)
    assert orc.overlap(E, 0.0) == 1.0
    al = [orc.overlap(E, d) for d in [0.0005, 0.001, 0.002, 0.004, 0.008]]
    assert all(x > y for x, y in zip(al, al[1:])) and 0 < al[-1] < al[0] < 1   # decreasing in dbeta
    # independent writing with numpy: alpha = mean(min(1, tau))
    tau = np.exp(-0.002 * E.astype(np.float64))
    tau /= tau.mean()
    assert abs(orc.overlap(E, 0.002) - np.minimum(1.0, tau).mean()) <= 1e-13
    # the adaptive step brackets the target
    for target in [0.95, 0.85, 0.6]:
        d = orc.adaptive_dbeta(E, target, 0.05)
        assert 0 < d < 0.05 and orc.overlap(E, d) >= target > orc.overlap(E, d * (1 + 1e-9) + 1e-12)
    assert orc.adaptive_dbeta(E, 0.01, 0.001) == 0.001          # dbeta_max already satisfies the target
    # inside the loop: steps shrink where the energy distribution is wide (critical region) -- PAPER.md:108
    pa = orc.OraclePA(16, 3000, seed=8)
    steps = []
    while pa.beta < 0.6 and len(steps) < 200:
        nb = pa.adaptive_beta(0.85, 0.05)
        steps.append(nb - pa.beta)
        pa.step(nb, 2)
    assert pa.beta >= 0.6 and min(steps) < 0.5 * max(steps)


# ---------------------------------------------------------------------------------------------------
# A5 scan / copy, A6 partitions
# ---------------------------------------------------------------------------------------------------
def test_scan_copy_parent_plain_definitions():
    rng = np.random.default_rng(11)
    L, R = 8, 5000
    n = rng.poisson(1.0, R).astype(np.uint32)
    n[100] = 700  # a heavy parent
    n[:10] = 0
    off, Rnew = orc.exclusive_scan(n)
    assert Rnew == int(n.sum()) and off[0] == 0 and off[-1] == Rnew
    assert np.array_equal(off[1:], np.cumsum(n.astype(np.int64)).astype(np.uint32))
    parent = orc.parent_of(n, off, Rnew)
    assert np.array_equal(parent, np.repeat(np.arange(R, dtype=np.uint32), n))
    src = rng.integers(0, 2 ** 32, (R, 2), dtype=np.uint64).astype(np.uint32)
    Es = rng.integers(-128, 128, R).astype(np.int32)
    Ms = rng.integers(-64, 64, R).astype(np.int32)
    dst, Ed, Md = orc.copy_population(L, n, off, src, Es, Ms, Rnew)
    assert np.array_equal(dst, src[parent]) and np.array_equal(Ed, Es[parent]) and np.array_equal(Md, Ms[parent])


@pytest.mark.parametrize("P", [1, 3, 148])
def test_partition_table_and_stats_invariants(P):
    rng = np.random.default_rng(P)
    R = 10007
    n = rng.poisson(1.0, R).astype(np.uint32)
    n[2000:2300] = 0
    n[5000] = 400
    off, Rnew = orc.exclusive_scan(n)
    old = orc.partition_table(R, P)
    new = orc.partition_table(Rnew, P)
    for tab, tot in [(old, R), (new, Rnew)]:
        cnt = np.diff(tab.astype(np.int64))
        assert tab[0] == 0 and tab[-1] == tot and cnt.max() - cnt.min() <= 1 and np.all(cnt >= 0)
        assert np.all(np.diff(cnt) <= 0)  # the larger partitions come first
    st, moved = orc.partition_stats(n, off, P, old, new)
    cnt, born, maxg, minl = st[:, 0].astype(np.int64), st[:, 1].astype(np.int64), st[:, 2], st[:, 3]
    assert born.sum() == Rnew and cnt.sum() == Rnew
    assert maxg.sum() == minl.sum()  # total excess = total shortage
    assert np.array_equal(np.maximum(born - cnt, 0), maxg) and np.array_equal(np.maximum(cnt - born, 0), minl)
    parent = np.repeat(np.arange(R), n)
    part_of_parent = np.searchsorted(old[1:], parent, side="right")
    part_of_child = np.searchsorted(new[1:], np.arange(Rnew), side="right")
    assert moved == int((part_of_parent != part_of_child).sum())
    assert np.array_equal(born, np.bincount(part_of_parent, minlength=P))
    if P == 1:
        assert moved == 0
    # fewer replicas than partitions
    tiny = orc.partition_table(5, 148)
    assert tiny[-1] == 5 and np.diff(tiny.astype(np.int64)).max() == 1


# ---------------------------------------------------------------------------------------------------
# A6b redistribution policies (readings G21-G23)
# ---------------------------------------------------------------------------------------------------
def test_policy_none_and_balanced_and_naive_closed_forms():
    rng = np.random.default_rng(5)
    for P in [1, 2, 8, 148]:
        born = rng.integers(0, 50000, P).astype(np.uint32)
        Rn = int(born.sum())
        cnt, _ = orc.policy_counts(born, orc.POLICY_NONE)
        assert np.array_equal(cnt, born)                      # nothing moves
        cnt, _ = orc.policy_counts(born, orc.POLICY_BALANCED)
        assert np.array_equal(cnt, np.diff(orc.partition_table(Rn, P).astype(np.int64)))
        cnt, _ = orc.policy_counts(born, orc.POLICY_NAIVE)
        assert int(cnt.sum()) == Rn
        pool = int((born // 2).sum())
        want = born.astype(np.int64) - born // 2 + pool // P + (np.arange(P) < pool % P)
        assert np.array_equal(cnt, want)
        # the excess over the mean halves (up to rounding): "relaxes fast to the flat behaviour"
        e0, e1 = born.astype(np.float64) - Rn / P, cnt.astype(np.float64) - Rn / P
        assert np.all(np.abs(e1 - e0 / 2) <= 1.0)


def test_policy_main_by_hand():
    # P = 3, B = 10, maxexc = 1 (window 10), R' = 90, r = (30, 30, 30)
    cnt, moves = orc.policy_counts([30, 35, 25], orc.POLICY_MAIN, 10, 1)
    assert cnt.tolist() == [30, 35, 25] and moves == 0          # everyone inside the window: nothing moves
    cnt, moves = orc.policy_counts([60, 20, 10], orc.POLICY_MAIN, 10, 1)
    # excess (30,-10,-20): 0->2 (50,20,20) e=(20,-10,-10); 0->1 [tie: lowest index] (40,30,20) e=(10,0,-10): stop
    assert cnt.tolist() == [40, 30, 20] and moves == 2
    cnt, moves = orc.policy_counts([60, 20, 10], orc.POLICY_MAIN, 10, 2)
    # window 20: (30,-10,-20): 0->2 gives (50,20,20) e=(20,-10,-10): stop after one move
    assert cnt.tolist() == [50, 20, 20] and moves == 1
    cnt, moves = orc.policy_counts([0, 0, 91], orc.POLICY_MAIN, 10, 1)
    # r = (31,30,30): e=(-31,-30,61): 2->0 (10,0,81) e=(-21,-30,51); 2->1 (10,10,71) e=(-21,-20,41); 2->0 (20,10,61)
    # e=(-11,-20,31); 2->1 (20,20,51) e=(-11,-10,21); 2->0 (30,20,41) e=(-1,-10,11); 2->1 (30,30,31) e=(-1,0,1): stop
    assert cnt.tolist() == [30, 30, 31] and moves == 6
    # block size 1, window 1: stops as soon as every |cnt - r| <= 1
    cnt, moves = orc.policy_counts([5, 1, 0], orc.POLICY_MAIN, 1, 1)
    assert cnt.tolist() == [3, 2, 1] and moves == 2  # r=(2,2,2), e=(3,-1,-2): 0->2, (4,1,1) e=(2,-1,-1): 0->1, (3,2,1) e=(1,0,-1): stop


def test_policy_main_ties_on_the_excess_side_by_hand():
    """reading G21 says "ties: lowest index" for the largest excess as well as for the largest shortage (PAPER.md:106
    defines only excess and shortage): cases where equal excesses share an odd number of moves, so that taking the LAST
    of the tied partitions instead ends with other counts"""
    from main_by_hand import MAIN_BY_HAND
    for born, B, maxexc, want, moves in MAIN_BY_HAND:
        cnt, mv = orc.policy_counts(born, orc.POLICY_MAIN, B, maxexc)
        assert cnt.tolist() == want and mv == moves, born


@pytest.mark.parametrize("P,B,maxexc", [(8, 1024, 1), (8, 1024, 2), (148, 1024, 1), (5, 1, 1), (16, 256, 3)])
def test_policy_main_invariants(P, B, maxexc):
    rng = np.random.default_rng(P * 7 + maxexc)
    for trial in range(30):
        scale = rng.choice([2000, 20480, 90000])
        born = (rng.gamma(2.0, scale / 2.0, P)).astype(np.uint32)
        Rn = int(born.sum())
        cnt, moves = orc.policy_counts(born, orc.POLICY_MAIN, B, maxexc)
        r = np.diff(orc.partition_table(Rn, P).astype(np.int64))
        c = cnt.astype(np.int64)
        assert int(c.sum()) == Rn and np.all(c >= 0)
        assert np.all(np.abs(c - r) <= maxexc * B)                     # everyone inside the window
        assert np.all((c - born.astype(np.int64)) % B == 0)            # replicas move in whole blocks
        inside = np.all(np.abs(born.astype(np.int64) - r) <= maxexc * B)
        assert (moves == 0) == bool(inside)                            # untouched iff already inside the window
        maxg, minl = np.maximum(c - r, 0), np.maximum(r - c, 0)
        assert maxg.sum() == minl.sum()
        assert np.array_equal(orc.starts_from_counts(cnt), np.concatenate([[0], np.cumsum(c)]).astype(np.uint32))


def test_policies_inside_the_pa_loop():
    # the policy only re-draws partition boundaries: populations, Q, counts are those of the default policy; the paper's
    # diagnostics follow their definitions
    ref = orc.OraclePA(8, 4096, P=8, seed=21)
    runs = {pol: orc.OraclePA(8, 4096, P=8, seed=21, policy=pol, block=64, maxexc=1)
            for pol in (orc.POLICY_MAIN, orc.POLICY_NAIVE, orc.POLICY_NONE)}
    for k in range(1, 13):
        ir = ref.step(0.04 * k, 1)
        for pol, pa in runs.items():
            info = pa.step(0.04 * k, 1)
            assert np.array_equal(pa.spins, ref.spins) and info["Q"] == ir["Q"] and np.array_equal(info["n"], ir["n"])
            st = info["part_stats"].astype(np.int64)
            cnt, born, maxg, minl = st[:, 0], st[:, 1], st[:, 2], st[:, 3]
            assert cnt.sum() == born.sum() == pa.R and maxg.sum() == minl.sum()
            assert np.array_equal(np.maximum(born - cnt, 0), maxg) and np.array_equal(np.maximum(cnt - born, 0), minl)
            assert np.array_equal(np.diff(info["part_start"].astype(np.int64)), cnt)
            if pol == orc.POLICY_NONE:
                assert np.array_equal(cnt, born) and info["moved"] == 0
            if pol == orc.POLICY_MAIN:
                r = np.diff(orc.partition_table(pa.R, 8).astype(np.int64))
                assert np.all(np.abs(cnt - r) <= 64)


# ---------------------------------------------------------------------------------------------------
# C4 Metropolis
# ---------------------------------------------------------------------------------------------------
def test_thresholds():
    mp.dps = 40
    for beta in [0.005, 0.3, 0.4407, 1.0, 2.5]:
        T4, T8 = orc.thresholds(beta)
        assert T4 == int(mp.floor(mpf(2) ** 32 * mp.exp(-4 * mpf(beta)))) or abs(
            T4 - int(mp.floor(mpf(2) ** 32 * mp.exp(-4 * mpf(beta))))) <= 1
        assert abs(T8 - int(mp.floor(mpf(2) ** 32 * mp.exp(-8 * mpf(beta))))) <= 1
        assert T8 < T4 < 2 ** 32
    assert orc.thresholds(0.0) == (2 ** 32 - 1, 2 ** 32 - 1)  # clamp (reading G10)
    assert orc.thresholds(50.0) == (0, 0)


def _pack_grid(L, g):
    return orc.pack(L, np.asarray(g, np.int8).reshape(-1))


def test_zero_temperature_dynamics_by_hand():
    L = 4
    N = L * L
    up = np.ones((L, L), np.int8)
    # (a) all-up is frozen: every site has a=0, dE=8, T8=0
    pop = np.stack([_pack_grid(L, up)])
    orc.sweeps(L, pop, 1, 1, 3, 0, 0)
    assert np.array_equal(orc.unpack(L, pop[0]), up.reshape(-1))
    # (b) one flipped spin heals (a=4 -> dE=-8 -> flip); its neighbours have a=1 -> dE=+4 -> stay (T4=0)
    for (y, x) in [(0, 0), (1, 2), (3, 3), (2, 1)]:
        g = up.copy()
        g[y, x] = -1
        pop = np.stack([_pack_grid(L, g)])
        orc.sweeps(L, pop, 5, 2, 1, 0, 0)
        assert np.array_equal(orc.unpack(L, pop[0]), up.reshape(-1))
    # (c) checkerboard: colour 0 is visited first, all its sites have a=4 and flip to the value of colour 1;
    #     then colour-1 sites have a=0 and stay  ->  uniform lattice equal to the colour-1 value
    yy, xx = np.divmod(np.arange(N), L)
    for c1val in [1, -1]:
        g = np.where((xx + yy) % 2 == 1, c1val, -c1val).astype(np.int8)
        pop = np.stack([orc.pack(L, g)])
        orc.sweeps(L, pop, 5, 2, 1, 0, 0)
        assert np.array_equal(orc.unpack(L, pop[0]), np.full(N, c1val, np.int8))
    # (d) dE = 0 always flips (reading G9): vertical stripes of width 1 on L=4: every site has a=2
    g = np.where(xx % 2 == 0, 1, -1).astype(np.int8)
    pop = np.stack([orc.pack(L, g)])
    orc.sweeps(L, pop, 5, 2, 1, 0, 0)
    # colour 0 flips everywhere (a=2); afterwards each colour-1 site sees: left/right flipped -> equal to it,
    # up/down unchanged colour-0?? no: up/down neighbours of a colour-1 site are colour 0 as well -> all four
    # neighbours flipped.  Before: a=2 (left/right anti, up/down aligned); after colour 0: left/right aligned,
    # up/down anti -> a=2 again -> flips.  Net effect of one sweep: global flip.
    assert np.array_equal(orc.unpack(L, pop[0]), -g)


def test_sweep_random_keying_on_all_up_lattice():
    # all-up lattice at finite beta: every colour-0 site has a=0, so it flips iff its keyed word < T8;
    # colour-0 sites are not touched again in the same sweep.  Predict with the big-int Philox.
    L, seed, step, slot_count = 8, 0xABCDEF0123456789, 12, 3
    T4, T8 = 0x9E3779B9, 0x3243F6A8  # synthetic thresholds with all 32 bits in play (p = 0.62, 0.20)
    pop = np.stack([orc.pack(L, np.ones(L * L, np.int8))] * slot_count)
    orc.sweeps(L, pop, seed, step, 1, T4, T8)
    for slot in range(slot_count):
        s = orc.unpack(L, pop[slot]).reshape(L, L)
        for y in range(L):
            for k in range(L // 2):
                x = 2 * k + (y & 1)  # colour 0
                w = philox_ref.sweep_word(seed, step, slot, 0, 0, y * (L // 2) + k)
                assert s[y, x] == (-1 if w < T8 else 1), (slot, y, x)
    # second sweep index t=1 uses counter word c2 = 2t+colour: all-up again, 2 sweeps, check t=1 is used:
    # (statistical) flips after 2 sweeps differ from after 1 sweep
    pop2 = np.stack([orc.pack(L, np.ones(L * L, np.int8))])
    orc.sweeps(L, pop2, seed, step, 2, T4, T8)
    assert not np.array_equal(pop2[0], pop[0])


@pytest.mark.parametrize("L", [16, 32])
def test_sweep_keying_groups_beyond_the_first_on_all_up_lattice(L):
    """DESIGN.md C3 (reading G20) for group index gamma > 0: L = 16 has 4 groups per half-sweep, L = 32 has 16, so the
    counter word c1 = 8*gamma + (b >> 2) is exercised for gamma up to 15.  All-up lattice: every colour-0 site has
    a = 0 and flips iff its keyed 32-bit uniform (big-integer writing, tests/philox_ref.py) is < T8."""
    seed, step = 0x0F1E2D3C4B5A6978, 7
    T4, T8 = 0x9E3779B9, 0x3243F6A8
    slots = [0, 5]
    pop = np.stack([orc.pack(L, np.ones(L * L, np.int8))] * 6)
    orc.sweeps(L, pop, seed, step, 1, T4, T8)
    half = L // 2
    for slot in slots:
        s = orc.unpack(L, pop[slot]).reshape(L, L)
        flips = 0
        for y in range(L):
            for k in range(half):
                x = 2 * k + (y & 1)  # colour 0
                w = philox_ref.sweep_word(seed, step, slot, 0, 0, y * half + k)
                assert s[y, x] == (-1 if w < T8 else 1), (slot, y, x)
                flips += w < T8
        assert 0.1 * L * half < flips < 0.3 * L * half  # p = T8 / 2^32 = 0.196: the pin is not vacuous


def _reference_metropolis(L, spins, seed, step, slot, theta, T4, T8):
    """C4 + C3 (reading G20) written a second time, from DESIGN.md's prose, on a +-1 numpy grid with the big-integer
    Philox of tests/philox_ref.py: sweep t = colour 0 then colour 1; active site ordinal q = y*(L/2) + k,
    x = 2k + ((y + colour) & 1); a = number of anti-aligned neighbours; flip iff a >= 2, or a == 1 and u < T4, or
    a == 0 and u < T8; u = philox_ref.sweep_word(seed, step, slot, t, colour, q)."""
    g = np.array(spins, np.int64).reshape(L, L).copy()
    half = L // 2
    for t in range(theta):
        for colour in (0, 1):
            for y in range(L):
                for k in range(half):
                    x = 2 * k + ((y + colour) & 1)
                    nb = (g[y, (x + 1) % L], g[y, (x - 1) % L], g[(y + 1) % L, x], g[(y - 1) % L, x])
                    a = sum(1 for v in nb if v != g[y, x])
                    u = philox_ref.sweep_word(seed, step, slot, t, colour, y * half + k)
                    if a >= 2 or (a == 1 and u < T4) or (a == 0 and u < T8):
                        g[y, x] = -g[y, x]
    return g.reshape(-1).astype(np.int8)


@pytest.mark.parametrize("L,beta", [(16, 0.3), (32, 0.44)])
def test_sweeps_whole_lattice_against_second_writing(L, beta):
    """Whole lattice after theta = 2 sweeps of random lattices == the independent writing above: fixes the keying of
    colour 1 (c2 = 2t + 1), of the second sweep (t = 1), of every group gamma, and the bit order of the uniform, for
    all three neighbour classes (random lattices have a = 0..4 sites)."""
    seed, step, theta = 0x1122334455667788 + L, 3, 2
    T4, T8 = orc.thresholds(beta)
    pop = orc.init_population(L, 3, seed)
    want = {slot: _reference_metropolis(L, orc.unpack(L, pop[slot]), seed, step, slot, theta, T4, T8) for slot in (0, 2)}
    orc.sweeps(L, pop, seed, step, theta, T4, T8)
    for slot, w in want.items():
        assert np.array_equal(orc.unpack(L, pop[slot]), w), slot
    # the same through the slot-list entry point with a slot index that is not the position in the list
    one = orc.init_population(L, 3, seed)[2:3].copy()
    orc.sweeps_slots(L, np.array([2], np.uint32), one, seed, step, theta, T4, T8)
    assert np.array_equal(orc.unpack(L, one[0]), want[2])


def test_sweeps_slots_equals_sweeps_and_slot_keying():
    L, R, seed, step = 8, 64, 77, 5
    pop = orc.init_population(L, R, seed)
    T4, T8 = orc.thresholds(0.4)
    a = pop.copy()
    orc.sweeps(L, a, seed, step, 3, T4, T8)
    slots = np.array([5, 0, 63, 17], np.uint32)
    b = pop[slots].copy()
    orc.sweeps_slots(L, slots, b, seed, step, 3, T4, T8)
    assert np.array_equal(b, a[slots])
    # a sub-range call equals the full call restricted to it
    c = pop.copy()
    orc.sweeps(L, c, seed, step, 3, T4, T8, first=10, count=20)
    assert np.array_equal(c[10:30], a[10:30]) and np.array_equal(c[:10], pop[:10])


def test_global_flip_covariance():
    # acceptance depends only on XORs of neighbouring spins and randoms are keyed by site:
    # the complemented population follows the complemented trajectory (SURVEY.md 8(c) Metropolis pin iii)
    L, R, seed = 16, 200, 2024
    pop = orc.init_population(L, R, seed)
    a = orc.OraclePA(L, R, seed=seed, spins=pop)
    b = orc.OraclePA(L, R, seed=seed, spins=~pop)
    for k in range(1, 6):
        ia = a.step(0.1 * k, 2)
        ib = b.step(0.1 * k, 2)
        assert ia["Q"] == ib["Q"] and np.array_equal(ia["n"], ib["n"])
        assert np.array_equal(a.spins, ~b.spins)
        assert np.array_equal(a.E, b.E) and np.array_equal(a.M, -b.M)


@pytest.mark.slow
def test_metropolis_samples_the_boltzmann_distribution_L4():
    # 40000 independent replicas of L=4, 60 sweeps at fixed beta from a uniform start: the energy histogram
    # must follow g(E) exp(-beta E) / Z (exact, brute force).  Pins acceptance rule + thresholds + RNG use.
    L, R, beta = 4, 40000, 0.35
    dos = {int(k): v for k, v in GOLD["dos_L4"].items()}
    pop = orc.init_population(L, R, 808)
    T4, T8 = orc.thresholds(beta)
    orc.sweeps(L, pop, 808, 1, 60, T4, T8)
    E, M = orc.energy_mag(L, pop)
    levels = sorted(dos)
    w = np.array([dos[e] * math.exp(-beta * e) for e in levels])
    p = w / w.sum()
    obs = np.array([(E == e).sum() for e in levels], float)
    keep = R * p >= 5
    chi2 = ((obs[keep] - R * p[keep]) ** 2 / (R * p[keep])).sum() + (obs[~keep].sum() - R * p[~keep].sum()) ** 2 / max(
        R * p[~keep].sum(), 1e-9)
    assert chi2 < stats.chi2.ppf(1 - 1e-6, keep.sum())
    assert abs(M.mean()) < 5 * M.std() / math.sqrt(R)  # Z2 symmetry


# ---------------------------------------------------------------------------------------------------
# whole PA loop against the exact partition function (eq. 3 + eq. 5, reading G1)
# ---------------------------------------------------------------------------------------------------
@pytest.mark.slow
def test_pa_lnZ_L4_large_population():
    L, R0, K = 4, 65536, 50
    pa = orc.OraclePA(L, R0, seed=4)
    sizes = []
    for k in range(1, K + 1):
        info = pa.step(k / K, 5)
        sizes.append(info["Rnew"])
        assert int(info["n"].sum()) == info["Rnew"] == pa.R
    exact = float(GOLD["lnZ"]["L4_beta1"])
    assert abs(pa.lnZ - exact) < 0.01, (pa.lnZ, exact)  # expect |delta| <~ 0.003
    z = (np.array(sizes) - R0) / math.sqrt(R0)  # R' ~ Poisson(R0) each step (reading G2)
    assert abs(z.mean()) < 5 / math.sqrt(K) and 0.6 < z.std() < 1.5
    assert max(sizes) <= pa.capacity


def test_pa_config1_lnZ_against_exact_L8():
    # BASELINE.json configs[0]: L=8, R=1024, seed 1, 100 uniform steps to beta=1, theta=10
    pa = orc.OraclePA(8, 1024, seed=1)
    for k in range(1, 101):
        pa.step(k * 0.01, 10)
        E, M = orc.energy_mag(8, pa.spins)
        assert np.array_equal(E, pa.E) and np.array_equal(M, pa.M)
    exact = float(GOLD["lnZ"]["L8_beta1"])
    assert abs(pa.lnZ - exact) < 0.2, (pa.lnZ, exact)  # run-to-run sd ~0.04
    obs = pa.observables()
    assert obs["mean_absM"] / 64 > 0.99  # ordered phase at beta = 1
    assert abs(obs["mean_E"] / 64 + 2) < 0.01


@pytest.mark.slow
def test_pa_lnZ_mean_over_seeds_L8():
    exact = float(GOLD["lnZ"]["L8_beta1"])
    vals = []
    for seed in range(100, 108):
        pa = orc.OraclePA(8, 1024, seed=seed)
        for k in range(1, 101):
            pa.step(k * 0.01, 10)
        vals.append(pa.lnZ - exact)
    vals = np.array(vals)
    assert abs(vals.mean()) < 4 * max(vals.std(ddof=1), 0.02) / math.sqrt(len(vals)) + 0.01, vals


def test_wrong_readings_of_eq5_are_far_off():
    # reading G1: without the logarithm, or with the opposite sign, the result is off by O(10..100)
    pa = orc.OraclePA(4, 4096, seed=3)
    sumQ = 0.0
    for k in range(1, 21):
        info = pa.step(k * 0.05, 3)
        sumQ += info["Q"]
    exact = float(GOLD["lnZ"]["L4_beta1"])
    assert abs(pa.lnZ - exact) < 0.3  # coarse schedule (dbeta=0.05, theta=3): statistical error ~0.05
    assert abs((pa.ln_omega + sumQ) - exact) > 5  # "sum of Q" reading
    assert abs((pa.ln_omega - pa.sum_lnQ) - exact) > 5  # opposite sign


def test_capacity_and_extinction_errors_leave_state_unchanged():
    pa = orc.OraclePA(8, 256, seed=9, capacity=256)
    before = pa.spins.copy()
    tries = 0
    with pytest.raises(orc.OracleError):
        for k in range(1, 200):  # R' ~ Poisson(256) exceeds 256 about half the time
            before, R_before = pa.spins.copy(), pa.R
            tries += 1
            pa.step(0.001 * k, 0)
    assert np.array_equal(pa.spins, before) and pa.R == R_before


# ---------------------------------------------------------------------------------------------------
# A8 observables
# ---------------------------------------------------------------------------------------------------
def test_moment_sums_exact_integers():
    rng = np.random.default_rng(3)
    R = 5000
    E = (4 * rng.integers(-8192, 8192, R)).astype(np.int32)
    M = rng.integers(-16384, 16385, R).astype(np.int32)
    M[:10] = 16384
    s = orc.moment_sums(E, M)
    Ei, Mi = [int(x) for x in E], [int(x) for x in M]
    assert s["sum_E"] == sum(Ei) and s["sum_E2"] == sum(e * e for e in Ei)
    assert s["sum_absM"] == sum(abs(m) for m in Mi) and s["sum_M2"] == sum(m * m for m in Mi)
    assert s["sum_M4"] == sum(m ** 4 for m in Mi)
    big = orc.moment_sums(np.zeros(300000, np.int32), np.full(300000, 16384, np.int32))
    assert big["sum_M4"] == 300000 * 16384 ** 4 > 2 ** 64  # needs the 128-bit accumulator


# ---------------------------------------------------------------------------------------------------
# heating protocol ("the cooling of the population and the heating of the population ... the initial
# temperature of heating is chosen close to zero temperature.  The initial value of the corresponding free energy was
# determined accordingly"): eq. 3 and eq. 5 with NEGATIVE dbeta (reading G29)
# ---------------------------------------------------------------------------------------------------
def test_heating_from_the_ground_states_reaches_the_exact_lnZ_L4():
    L, N, R0, beta0 = 4, 16, 30000, 2.0
    dos, _ = exact_ising.brute_force_dos(L)
    lnZ0 = float(exact_ising.lnZ_from_dos(dos, beta0))          # ln Omega of the heating run, "determined accordingly"
    assert abs(lnZ0 - (math.log(2.0) + 2 * N * beta0)) < 1e-5    # two ground states of energy -2N; excitations ~ 16 e^-16
    up = orc.pack(L, np.ones(N, np.int8))
    down = orc.pack(L, -np.ones(N, np.int8))
    spins = np.stack([up if j % 2 == 0 else down for j in range(R0)])
    pa = orc.OraclePA(L, R0, seed=21, beta0=beta0, spins=spins)
    betas = [beta0 - 0.05 * k for k in range(1, 37)]             # 2.0 -> 0.2
    for b in betas:
        info = pa.step(b, 5)
        assert info["dbeta"] < 0 and info["Q"] < 1.0   # E < 0 throughout: weights exp(-dbeta E) < 1
    lnZ = lnZ0 + pa.sum_lnQ
    exact = float(exact_ising.lnZ_from_dos(dos, betas[-1]))
    assert abs(lnZ - exact) < 0.03, (lnZ, exact)
    # and the population has left the ground states: <E> at beta = 0.2 from the density of states
    Es = np.array([int(k) for k in dos.keys()], float)
    g = np.array([float(v) for v in dos.values()])
    w = g * np.exp(-betas[-1] * Es)
    assert abs(pa.E.mean() - (w * Es).sum() / w.sum()) < 0.25


# ---------------------------------------------------------------------------------------------------
# A4c systematic resampling (PAPER.md:54 -> ref. [3]; reading G30)
# ---------------------------------------------------------------------------------------------------
def test_systematic_resampling_against_a_big_integer_writing_and_its_laws():
    rng = np.random.default_rng(11)
    seed = 0xABCDEF0123
    for step, R in [(1, 1), (2, 7), (3, 1000), (9, 4097)]:
        tau = np.exp(rng.normal(0.0, 1.2, R))
        tau *= R / tau.sum()
        scale = 0.97
        n = orc.systematic_counts(tau, scale, seed, step)
        # second writing: Python integers, U from the big-integer Philox (counter (0, 0, 1, tag 1 | step), word 0)
        U = philox_ref.keyed(seed, 0, 0, 1, 1, step)[0]
        assert orc.systematic_uniform(seed, step) == U
        lam = [float(t) * scale for t in tau]
        Lam = [int(math.floor(x * 4294967296.0)) for x in lam]
        C, ref = 0, []
        for L_ in Lam:
            ref.append(((C + L_ + U) >> 32) - ((C + U) >> 32))
            C += L_
        assert [int(x) for x in n] == ref
        # laws: n_j is floor or ceil of Lam_j / 2^32; the population is floor(sum Lam / 2^32) or that + 1
        for nj, L_ in zip(ref, Lam):
            assert nj in (L_ >> 32, (L_ >> 32) + 1)
        assert sum(ref) in (C >> 32, (C >> 32) + 1)
        assert abs(sum(ref) - sum(lam)) < 1.0 + R * 2.0 ** -32
    # equal unit weights: every parent has exactly one child whatever U is
    assert np.all(orc.systematic_counts(np.ones(500), 1.0, 5, 1) == 1)
    assert np.all(orc.systematic_counts(np.zeros(10), 1.0, 5, 1) == 0)
    # E[n_j] = lambda_j: U runs over the steps; a parent with lambda = 0.3 gets a child in 30 % of the steps
    tau = np.array([0.3, 1.7, 2.0, 0.25, 3.75])
    acc = np.zeros(5)
    K = 4000
    for step in range(1, K + 1):
        acc += orc.systematic_counts(tau, 1.0, 77, step)
    assert np.all(np.abs(acc / K - tau) < 4 * np.sqrt(0.25 / K))
    assert acc[2] == 2 * K  # integer lambda: deterministic


def test_pa_with_systematic_resampling_keeps_the_population_and_gets_lnZ_right():
    L = 8
    pa = orc.OraclePA(L, 4096, seed=5, rule=orc.RULE_SYSTEMATIC)
    for k in range(1, 41):
        pa.step(0.025 * k, 3)
        assert abs(pa.R - 4096) <= 1  # sum lambda = R0 up to rounding: the population stays at R0
    exact = float(exact_ising.kaufman_lnZ(L, 1.0))
    assert abs(pa.lnZ - exact) < 0.3, (pa.lnZ, exact)
