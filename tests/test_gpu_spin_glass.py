"""GPU parity (-m gpu) of the second Hamiltonian, the 2D +-J spin glass (pa_set_bonds, pa_overlap_hist; D1,
SURVEY.md 8(f)-4), through the C ABI against oracle/pa_oracle.c section D1 on the same seeded samples.
Same bar as tests/test_gpu_parity.py: integers bit-exact, Q / tau / ln Z to 1e-12."""
import numpy as np
import pytest

from oracle import pa_oracle as orc
from paper_2006_00561_b200 import inputs

from test_gpu_parity import RTOL, _binding, compare_population, lockstep, make_pair, rel

pytestmark = pytest.mark.gpu


def sample_with_parity(L, seed, odd):
    """a +-J sample whose number of negative bonds is odd (E = 2 mod 4) or even (E = 0 mod 4)"""
    for s in range(seed, seed + 64):
        Jx, Jy = inputs.bond_sample(L, s)
        if (int((Jx < 0).sum() + (Jy < 0).sum()) & 1) == int(odd):
            return Jx, Jy
    raise AssertionError("no sample found")


@pytest.mark.parametrize("L,R0,odd", [(8, 700, 1), (8, 333, 0), (16, 500, 1), (32, 400, 0), (32, 257, 1), (64, 150, 1),
                                       (64, 97, 0), (128, 40, 1), (128, 33, 0)])
def test_initial_energies_and_lockstep(L, R0, odd):
    bonds = sample_with_parity(L, 10 * L + odd, odd)
    gpu, ora = make_pair(L, R0, 3, seed=40 + L, bonds=bonds)
    E, _ = gpu.energies()
    assert np.all(E % 4 == 2 * odd)
    compare_population(gpu, ora, "init")
    # reading G11: |dbeta| * 2N < 700, so the larger lattices take smaller temperature steps
    betas = {64: [0.06 * k for k in range(1, 8)], 128: [0.02 * k for k in range(1, 8)]}.get(L, [0.1, 0.25, 0.4, 0.6, 0.8, 1.0, 1.3])
    lockstep(gpu, ora, betas, theta=2)
    assert rel(gpu.log_Z()["lnZ"], ora.lnZ) <= RTOL


def test_structured_population_resample_only_and_policies():
    L, R0 = 32, 3000
    bonds = sample_with_parity(L, 5, 1)
    spins = inputs.structured_population(L, R0, 77)
    gpu, ora = make_pair(L, R0, 7, seed=8, spins=spins, bonds=bonds, policy=1, block=64, maxexc=1)
    lockstep(gpu, ora, [0.02, 0.05], theta=0)      # a6 by k_copy
    lockstep(gpu, ora, [0.08, 0.12], theta=1)      # a6 by the sweep's gather-on-load


def test_nearest_rule_and_adaptive_step_with_odd_sample():
    L, R0 = 16, 2000
    bonds = sample_with_parity(L, 90, 1)
    gpu, ora = make_pair(L, R0, 2, seed=3, bonds=bonds, rule=1)
    beta = 0.0
    for _ in range(5):
        b_gpu = gpu.adaptive_beta(0.85, 0.2)
        b_ora = ora.adaptive_beta(0.85, 0.2)
        assert abs(b_gpu - b_ora) <= 1e-9 * max(abs(b_ora), 1e-3)
        assert b_gpu > beta
        lockstep(gpu, ora, [b_gpu], theta=2)
        beta = b_gpu


def test_mattis_sample_shadows_the_ferromagnet_on_the_device():
    b = _binding()
    L, R0 = 64, 256
    Jx, Jy, eps = inputs.mattis_bonds(L, 4)
    ferro = b.PopulationAnnealer(L, R0, P=1, seed=21)
    glass = b.PopulationAnnealer(L, R0, P=1, seed=21)
    s0 = ferro.spins()
    eps_words = inputs.pack_pm1(eps)               # sigma -> eps * sigma: flip the bits where eps = -1
    glass.set_spins(s0 ^ ~eps_words[None, :])
    glass.set_bonds(inputs.pack_pm1(Jx), inputs.pack_pm1(Jy))
    for k in range(1, 7):
        ferro.step(0.08 * k, 3)
        glass.step(0.08 * k, 3)
        assert np.array_equal(ferro.energies()[0], glass.energies()[0])
        assert np.array_equal(glass.spins(), ferro.spins() ^ ~eps_words[None, :])
    assert ferro.log_Z()["lnZ"] == glass.log_Z()["lnZ"]


def test_full_block_population_sampled_slots_L64():
    L, R0 = 64, 1 << 16
    bonds = sample_with_parity(L, 400, 1)
    gpu, ora = make_pair(L, R0, 148, seed=12, bonds=bonds)
    lockstep(gpu, ora, [0.08, 0.16, 0.24, 0.3], theta=3, sweep_slots=600)


def test_set_bonds_rules_and_back_to_the_ferromagnet():
    b = _binding()
    L, R0 = 16, 64
    Jx, Jy = inputs.bond_sample(L, 1)
    px, py = inputs.pack_pm1(Jx), inputs.pack_pm1(Jy)
    gpu = b.PopulationAnnealer(L, R0, seed=5)
    E_ferro, _ = gpu.energies()
    with pytest.raises(b.PaError) as e:
        gpu._check(gpu._lib.pa_set_bonds(gpu._ctx, px.ctypes.data, None))
    assert e.value.code == b.PA_EINVAL
    gpu.set_bonds(px, py)
    assert np.array_equal(gpu.energies()[0], orc.energy_mag(L, gpu.spins(), (Jx, Jy))[0])
    gpu.set_bonds(None, None)
    assert np.array_equal(gpu.energies()[0], E_ferro)
    ones = np.ones(L * L, np.int8)
    gpu.set_bonds(inputs.pack_pm1(ones), inputs.pack_pm1(ones))   # all ferromagnetic through the +-J kernels
    assert np.array_equal(gpu.energies()[0], E_ferro)
    gpu.step(0.1, 1)
    with pytest.raises(b.PaError) as e:
        gpu.set_bonds(px, py)
    assert e.value.code == b.PA_EINVAL


@pytest.mark.parametrize("L,R0", [(8, 1001), (16, 700), (32, 512), (64, 333), (128, 70)])
def test_overlap_histogram(L, R0):
    bonds = sample_with_parity(L, 3 * L, 0)
    gpu, ora = make_pair(L, R0, 1, seed=L, bonds=bonds)
    assert np.array_equal(gpu.overlap_hist(), orc.overlap_hist(L, ora.spins))
    for k in (1, 2, 3):
        gpu.step(k * (0.02 if L == 128 else 0.08), 2)
    h = gpu.overlap_hist()
    assert np.array_equal(h, orc.overlap_hist(L, gpu.spins()))
    assert int(h.sum()) == gpu.R // 2


def test_overlap_histogram_large_population_ising():
    b = _binding()
    gpu = b.PopulationAnnealer(32, 1 << 17, seed=2)
    gpu.run([0.2, 0.4], 2)
    assert np.array_equal(gpu.overlap_hist(), orc.overlap_hist(32, gpu.spins()))


@pytest.mark.parametrize("world,L,theta", [(2, 32, 2), (3, 64, 1), (4, 16, 0)])
def test_sharded_ranks_with_bonds_equal_the_single_context(world, L, theta):
    """multi-GPU protocol (ranks emulated on one device) with the second Hamiltonian: every rank sets the same sample"""
    b = _binding()
    from paper_2006_00561_b200 import dist
    R0, seed = 1500, 60 + L
    Jx, Jy = sample_with_parity(L, 7 * L, 1)
    px, py = inputs.pack_pm1(Jx), inputs.pack_pm1(Jy)
    single = b.PopulationAnnealer(L, R0, P=1, seed=seed)
    single.set_bonds(px, py)
    sh = dist.ShardedAnnealer(L, R0, seed=seed, emulate=world, bonds=(px, py))
    E0 = np.concatenate([s_.energies()[0] for s_ in sh.shards])
    assert np.array_equal(E0, single.energies()[0]) and np.all(E0 % 4 == 2)
    dbeta = min(0.06, 600.0 / (2 * L * L))
    for k in range(1, 6):
        single.step(dbeta * k, theta)
        obs = sh.step(dbeta * k, theta)
        assert np.array_equal(sh.gather_spins(), single.spins()), k
        assert sum(o["sum_E"] for o in obs) == single.observables()["sum_E"]
        assert np.array_equal(np.concatenate([s_.energies()[0] for s_ in sh.shards]), single.energies()[0])
        for s_ in sh.shards:
            assert rel(s_.log_Z()["lnZ"], single.log_Z()["lnZ"]) <= RTOL


def test_set_spins_after_set_bonds_and_device_getters():
    """the test hook pa_set_spins recomputes E under the Hamiltonian in force; pa_energies with a device destination
    carries the energy offset of an odd sample too"""
    b = _binding()
    L, R = 32, 777
    Jx, Jy = sample_with_parity(L, 1234, 1)
    gpu = b.PopulationAnnealer(L, R, seed=8, capacity=4096)
    gpu.set_bonds(inputs.pack_pm1(Jx), inputs.pack_pm1(Jy))
    pop = inputs.structured_population(L, 1500, 3)
    gpu.set_spins(pop)
    Eo, Mo = orc.energy_mag(L, pop, (Jx, Jy))
    E, M = gpu.energies()
    assert gpu.R == 1500 and np.array_equal(E, Eo) and np.array_equal(M, Mo) and np.all(E % 4 == 2)
    Ed, Md = gpu.energies_device()
    assert np.array_equal(Ed.cpu().numpy(), Eo) and np.array_equal(Md.cpu().numpy(), Mo)
    assert gpu.observables()["sum_E"] == int(Eo.astype(np.int64).sum())
