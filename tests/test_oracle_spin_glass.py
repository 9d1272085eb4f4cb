"""Pins for the oracle's second Hamiltonian (-m "not gpu"): the 2D +-J spin glass, oracle/pa_oracle.c section D1
(readings G27, G28).  The paper gives no numbers for it, so the pins are what
the mathematics fixes: a second (vectorised numpy) writing of the energy on all 2^16 states of L = 4, the parity law of
E, gauge covariance (a Mattis sample J_ij = eps_i eps_j IS the ferromagnet, whose sweeps and ln Z are pinned in
tests/test_oracle_pins.py), hand-worked zero-temperature moves around single negative bonds, the Boltzmann
distribution and ln Z of a frustrated sample against exact enumeration, and numpy for the overlap histogram."""
import math

import numpy as np
import pytest
from scipy import stats

from oracle import pa_oracle as orc
from paper_2006_00561_b200 import inputs


def np_energy(L, s, Jx, Jy):
    """H = -sum_<ij> J_ij s_i s_j, second writing: s (..., L, L) +-1, bonds to the right (Jx) and below (Jy)"""
    s = s.astype(np.int64)
    jx, jy = Jx.reshape(L, L).astype(np.int64), Jy.reshape(L, L).astype(np.int64)
    return -(jx * s * np.roll(s, -1, axis=-1)).sum(axis=(-2, -1)) - (jy * s * np.roll(s, -1, axis=-2)).sum(axis=(-2, -1))


def all_states(L):
    N = L * L
    idx = np.arange(1 << N, dtype=np.uint32)
    bits = (idx[:, None] >> np.arange(N, dtype=np.uint32)[None, :]) & 1
    return (2 * bits.astype(np.int8) - 1).reshape(-1, L, L)


def packed_from_pm1(L, s):
    return np.stack([orc.pack(L, x.reshape(-1)) for x in s])


def unpack_all(L, packed):
    return np.stack([orc.unpack(L, w) for w in packed])


@pytest.mark.parametrize("seed", [11, 12, 13])
def test_energy_on_all_states_of_L4_equals_numpy_writing(seed):
    L = 4
    Jx, Jy = inputs.bond_sample(L, seed)
    S = all_states(L)
    ref = np_energy(L, S, Jx, Jy)
    packed = np.array([[i] for i in range(1 << 16)], np.uint32)  # L = 4: the 16 bits of the state index (layout C2)
    E, M = orc.energy_mag(L, packed, bonds=(Jx, Jy))
    assert np.array_equal(E, ref)
    assert np.array_equal(M, S.reshape(-1, 16).sum(axis=1))
    # parity law: E = 2u - 2N, u = #negative bonds (mod 2)  =>  E = 2 * (#negative) (mod 4)
    nneg = int((Jx < 0).sum() + (Jy < 0).sum())
    assert np.all((E - 2 * nneg) % 4 == 0)
    assert E.min() >= -2 * L * L and E.max() <= 2 * L * L


def test_parity_law_covers_both_classes():
    seen = set()
    for seed in range(20):
        Jx, Jy = inputs.bond_sample(8, 100 + seed)
        nneg = int((Jx < 0).sum() + (Jy < 0).sum())
        pop = inputs.random_packed_population(8, 64, seed)
        E, _ = orc.energy_mag(8, pop, bonds=(Jx, Jy))
        assert np.all((E - 2 * nneg) % 4 == 0)
        seen.add(nneg & 1)
    assert seen == {0, 1}


@pytest.mark.parametrize("L", [8, 16, 32])
def test_all_ferromagnetic_bonds_are_eq6(L):
    ones = np.ones(L * L, np.int8)
    pop = inputs.random_packed_population(L, 50, L)
    assert np.array_equal(orc.energy_mag(L, pop, bonds=(ones, ones))[0], orc.energy_mag(L, pop)[0])
    a, b = pop.copy(), pop.copy()
    T4, T8 = orc.thresholds(0.3)
    orc.sweeps(L, a, 5, 2, 3, T4, T8)
    orc.sweeps(L, b, 5, 2, 3, T4, T8, bonds=(ones, ones))
    assert np.array_equal(a, b)


@pytest.mark.parametrize("L", [8, 16, 32])
def test_mattis_sample_is_the_ferromagnet_under_the_gauge(L):
    """J_ij = eps_i eps_j:  E_J(eps sigma) = E_ferro(sigma), and -- the randoms being keyed by site and slot, the rule
    depending on a only -- sweeps_J(eps sigma) = eps * sweeps_ferro(sigma): ties section D1 to the pinned C4 sweeps."""
    Jx, Jy, eps = inputs.mattis_bonds(L, 7 + L)
    pop = inputs.random_packed_population(L, 40, 3 * L, p_up=0.7)
    s = unpack_all(L, pop)
    gs = packed_from_pm1(L, s * eps[None, :])
    assert np.array_equal(orc.energy_mag(L, gs, bonds=(Jx, Jy))[0], orc.energy_mag(L, pop)[0])
    T4, T8 = orc.thresholds(0.35)
    ferro = pop.copy()
    orc.sweeps(L, ferro, 9, 4, 3, T4, T8)
    orc.sweeps(L, gs, 9, 4, 3, T4, T8, bonds=(Jx, Jy))
    assert np.array_equal(unpack_all(L, gs), unpack_all(L, ferro) * eps[None, :])
    assert not np.array_equal(ferro, pop)


@pytest.mark.parametrize("L", [8, 16])
def test_gauge_covariance_of_a_frustrated_sample(L):
    Jx, Jy = inputs.bond_sample(L, 21 + L)
    rng = np.random.default_rng(5)
    eps = np.where(rng.random((L, L)) < 0.5, -1, 1).astype(np.int8)
    Jx2 = (Jx.reshape(L, L) * eps * np.roll(eps, -1, axis=1)).reshape(-1)
    Jy2 = (Jy.reshape(L, L) * eps * np.roll(eps, -1, axis=0)).reshape(-1)
    pop = inputs.random_packed_population(L, 30, 77)
    s = unpack_all(L, pop)
    gpop = packed_from_pm1(L, s * eps.reshape(-1)[None, :])
    assert np.array_equal(orc.energy_mag(L, pop, bonds=(Jx, Jy))[0], orc.energy_mag(L, gpop, bonds=(Jx2, Jy2))[0])
    T4, T8 = orc.thresholds(0.5)
    a, b = pop.copy(), gpop.copy()
    orc.sweeps(L, a, 1, 1, 2, T4, T8, bonds=(Jx, Jy))
    orc.sweeps(L, b, 1, 1, 2, T4, T8, bonds=(Jx2, Jy2))
    assert np.array_equal(unpack_all(L, b), unpack_all(L, a) * eps.reshape(-1)[None, :])


def test_hand_worked_negative_bonds_at_zero_temperature():
    """all-up 8 x 8 lattice, T4 = T8 = 0 (only dE <= 0 moves).
    (i) one negative bond Jx(3,2): E = -2N + 2; its two ends have a = 1 (dE = 4): nothing ever moves.
    (ii) Jx(3,2) and Jy(3,2) negative: E = -2N + 4; site (3,2) has a = 2 (dE = 0, always flips, reading G9); it is a
    colour-1 site, its neighbours (colour 0, visited first) have a = 1 and stay; after its flip it has a = 2 again
    (now through its two positive bonds), so sweep 2 flips it back: theta = 1 -> only (3,2) down, theta = 2 -> all up.
    (iii) all four bonds of (3,2) negative: a = 4 there (dE = -8) and a = 1 at its neighbours; it flips once, after which
    every bond is satisfied (E = -2N) and the lattice is frozen."""
    L, N = 8, 64
    up = orc.pack(L, np.ones(N, np.int8))[None, :].copy()
    site = 2 * L + 3

    def run(neg, theta):
        Jx, Jy = np.ones(N, np.int8), np.ones(N, np.int8)
        for kind, b in neg:
            (Jx if kind == "x" else Jy)[b] = -1
        E0 = orc.energy_mag(L, up, bonds=(Jx, Jy))[0][0]
        p = up.copy()
        orc.sweeps(L, p, 3, 1, theta, 0, 0, bonds=(Jx, Jy))
        return E0, orc.unpack(L, p[0]), orc.energy_mag(L, p, bonds=(Jx, Jy))[0][0]

    E0, s, E1 = run([("x", site)], 3)
    assert E0 == -2 * N + 2 and np.all(s == 1) and E1 == E0
    E0, s, E1 = run([("x", site), ("y", site)], 1)
    expect = np.ones(N, np.int8)
    expect[site] = -1
    assert E0 == -2 * N + 4 and np.array_equal(s, expect) and E1 == E0
    E0, s, E1 = run([("x", site), ("y", site)], 2)
    assert np.all(s == 1)
    E0, s, E1 = run([("x", site), ("y", site), ("x", site - 1), ("y", site - L)], 4)
    assert E0 == -2 * N + 8 and np.array_equal(s, expect) and E1 == -2 * N


def exact_dos(L, Jx, Jy):
    E = np_energy(L, all_states(L), Jx, Jy)
    vals, cnt = np.unique(E, return_counts=True)
    return vals, cnt


def test_boltzmann_distribution_of_a_frustrated_sample_L4():
    """detailed balance with the right dE: energy histogram after many sweeps == g(E) exp(-beta E) / Z by enumeration"""
    L, beta, R = 4, 0.45, 40000
    Jx, Jy = inputs.bond_sample(L, 31)
    vals, cnt = exact_dos(L, Jx, Jy)
    assert len(vals) > 4 and vals.min() > -2 * L * L  # frustrated: the ground state leaves bonds unsatisfied
    w = cnt * np.exp(-beta * (vals - vals.min()))
    p = w / w.sum()
    pop = orc.init_population(L, R, 17)
    T4, T8 = orc.thresholds(beta)
    orc.sweeps(L, pop, 17, 1, 60, T4, T8, bonds=(Jx, Jy))
    E, _ = orc.energy_mag(L, pop, bonds=(Jx, Jy))
    obs = np.array([(E == v).sum() for v in vals], float)
    keep = p * R >= 5
    o = np.append(obs[keep], obs[~keep].sum())
    e = np.append(p[keep] * R, p[~keep].sum() * R)
    if e[-1] == 0:
        o, e = o[:-1], e[:-1]
    chi2 = ((o - e) ** 2 / e).sum()
    assert chi2 < stats.chi2.ppf(1 - 1e-6, len(e) - 1), (chi2, len(e))


def test_pa_lnZ_of_a_frustrated_sample_against_enumeration_L4():
    """eq. 3 + eq. 5 with the +-J energies: ln Z(beta = 1) of one frustrated 4 x 4 sample (odd number of negative bonds,
    so E = 2 mod 4) against the sum over all 65 536 states"""
    L = 4
    for seed in range(40, 60):
        Jx, Jy = inputs.bond_sample(L, seed)
        if ((Jx < 0).sum() + (Jy < 0).sum()) % 2 == 1:
            break
    vals, cnt = exact_dos(L, Jx, Jy)
    assert vals[0] % 4 == 2
    exact = math.log(float((cnt * np.exp(-1.0 * (vals - vals.min()))).sum())) - vals.min()
    pa = orc.OraclePA(L, 1 << 15, seed=3, bonds=(Jx, Jy))
    for k in range(1, 21):
        pa.step(k * 0.05, 5)
    assert abs(pa.lnZ - exact) < 0.03, (pa.lnZ, exact)
    assert np.array_equal(pa.E, orc.energy_mag(L, pa.spins, bonds=(Jx, Jy))[0])


def test_pa_run_on_a_mattis_sample_shadows_the_ferromagnetic_run():
    """whole loop: with J = eps eps and the gauge-transformed initial population every E_j, hence Q, tau, the keyed copy
    counts and the keyed sweeps, equal the ferromagnet's step by step; populations stay related by eps"""
    L, R0 = 8, 512
    Jx, Jy, eps = inputs.mattis_bonds(L, 2)
    ferro = orc.OraclePA(L, R0, seed=9)
    start = packed_from_pm1(L, unpack_all(L, ferro.spins) * eps[None, :])
    glass = orc.OraclePA(L, R0, seed=9, spins=start, bonds=(Jx, Jy))
    for k in range(1, 13):
        a = ferro.step(0.05 * k, 2)
        b = glass.step(0.05 * k, 2)
        assert a["Q"] == b["Q"] and np.array_equal(a["n"], b["n"])
        assert np.array_equal(ferro.E, glass.E)
    assert ferro.lnZ == glass.lnZ
    assert np.array_equal(unpack_all(L, glass.spins), unpack_all(L, ferro.spins) * eps[None, :])


@pytest.mark.parametrize("L,R", [(8, 10), (8, 11), (16, 64), (32, 7)])
def test_overlap_histogram_equals_numpy(L, R):
    N = L * L
    pop = inputs.random_packed_population(L, R, 5 * L + R, p_up=0.6)
    bits = np.unpackbits(pop.view(np.uint8), axis=1, bitorder="little")[:, :N].astype(np.int64)
    s = 2 * bits - 1
    half = R // 2
    q = (s[:half] * s[half:2 * half]).sum(axis=1)
    ref = np.bincount((q + N) // 2, minlength=N + 1)
    h = orc.overlap_hist(L, pop)
    assert np.array_equal(h.astype(np.int64), ref) and int(h.sum()) == half


def test_overlap_of_identical_and_opposite_halves():
    L, N = 8, 64
    pop = inputs.random_packed_population(L, 6, 1)
    same = np.concatenate([pop, pop])
    h = orc.overlap_hist(L, same)
    assert h[N] == 6 and h.sum() == 6
    opp = np.concatenate([pop, ~pop])
    h = orc.overlap_hist(L, opp)
    assert h[0] == 6 and h.sum() == 6
