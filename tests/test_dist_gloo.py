"""world_size-2 gloo test (CPU) of bench.py's multi-process plumbing: barrier, max-over-ranks time, summed units.
The path itself does not shard ("replicas only"): each rank runs an independent replica, here the CPU oracle on a
tiny workload stands in for the per-rank work so that the aggregation is exercised end to end."""
import os
import socket

import pytest
import torch.multiprocessing as mp

from main_by_hand import MAIN_BY_HAND


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    os.environ.update({"RANK": str(rank), "WORLD_SIZE": str(world), "LOCAL_RANK": str(rank),
                       "MASTER_ADDR": "127.0.0.1", "MASTER_PORT": str(port)})
    from paper_2006_00561_b200 import dist
    from oracle import pa_oracle as orc
    g = dist.init_from_env(backend="gloo", device_kind="cpu")
    orc.set_threads(1)
    pa = orc.OraclePA(8, 64, seed=100 + rank)  # independent replica per rank
    dist.barrier(g)
    units = 0
    for k in range(1, 4):
        pa.step(0.1 * k, 2)
        units += 2 * 64 * pa.R
    seconds = 1.0 + rank  # synthetic per-rank time: the slowest rank must define the job time
    value, total, tmax = dist.aggregate_throughput(g, units, seconds)
    dist.barrier(g)
    q.put((rank, units, value, total, tmax, g.is_main))
    dist.shutdown(g)


def test_two_rank_aggregation_gloo():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, u0, v0, t0, m0, main0), (r1, u1, v1, t1, m1, main1) = res
    assert main0 and not main1
    assert t0 == t1 == u0 + u1 and m0 == m1 == 2.0  # max over ranks, not the mean
    assert v0 == v1 == pytest.approx((u0 + u1) / 2.0)


def test_single_process_is_identity():
    from paper_2006_00561_b200 import dist
    g = dist.Group()
    assert dist.aggregate_throughput(g, 10.0, 2.0) == (5.0, 10.0, 2.0)
    dist.barrier(g)


# ---------------------------------------------------------------------------------------------------
# partitioned redistribution, rank = partition
# ---------------------------------------------------------------------------------------------------
def test_exchange_plan_against_the_oracle_policies_and_its_invariants():
    """pa_dist_exchange_plan is a pure host function of the product library (no GPU needed): its partition counts must be
    the oracle's policy counts with born_p = T_p, and its slices must tile both sides exactly"""
    import numpy as np
    from oracle import pa_oracle as orc
    from paper_2006_00561_b200 import binding
    rng = np.random.default_rng(8)
    for world in [1, 2, 3, 8, 64]:
        for policy, block, maxexc in [(0, 1024, 1), (1, 1024, 1), (1, 64, 2), (2, 1024, 1), (3, 1024, 1)]:
            T = rng.integers(0, 60000, world).astype(np.int64)
            T[rng.integers(0, world)] = 0  # a rank without offspring
            if T.sum() == 0:
                T[0] = 5
            ns, base, counts = binding.exchange_plan(T, policy, block, maxexc)
            cnt, _ = orc.policy_counts(T.astype(np.uint32), policy, block, maxexc)
            assert np.array_equal(np.diff(ns), cnt.astype(np.int64)), (world, policy)
            assert np.array_equal(np.diff(base), T) and ns[-1] == base[-1] == T.sum()
            assert np.array_equal(counts.sum(axis=1), T)            # every child is sent exactly once
            assert np.array_equal(counts.sum(axis=0), np.diff(ns))  # every new slot is filled exactly once
            # order preserving: the destinations of a source's slices are non-decreasing, and so are the sources of a destination's
            for src in range(world):
                nz = np.nonzero(counts[src])[0]
                assert np.all(np.diff(nz) == 1) or len(nz) <= 1     # contiguous block of destinations
            if policy == 3:
                assert np.array_equal(counts, np.diag(T))           # nothing crosses a rank boundary
    with pytest.raises(binding.PaError) as ei:
        binding.exchange_plan([0, 0, 0])
    assert ei.value.code == binding.PA_EEXTINCT
    with pytest.raises(binding.PaError) as ei:
        binding.exchange_plan([5, -1, 3])
    assert ei.value.code == binding.PA_ECAPACITY


def test_main_policy_ties_on_the_excess_side_by_hand():
    """the same hand-worked cases through the oracle's policy function and through the product's host plan: two writings
    of reading G21, each pinned to the moves written out above rather than to one another"""
    import numpy as np
    from oracle import pa_oracle as orc
    from paper_2006_00561_b200 import binding
    for born, B, maxexc, want, moves in MAIN_BY_HAND:
        cnt, mv = orc.policy_counts(np.asarray(born, np.uint32), orc.POLICY_MAIN, B, maxexc)
        assert cnt.tolist() == want and mv == moves, ("oracle", born)
        ns, base, counts = binding.exchange_plan(born, binding.PA_POLICY_MAIN, B, maxexc)
        assert np.diff(ns).tolist() == want, ("plan", born)
        assert np.diff(base).tolist() == born
        # children keep their global order: rank dst receives the global range [ns[dst], ns[dst+1]) cut at the sources' ends
        for src in range(len(born)):
            for dst in range(len(born)):
                lo, hi = max(base[src], ns[dst]), min(base[src + 1], ns[dst + 1])
                assert counts[src, dst] == max(0, hi - lo)


def test_exchange_plan_invariants_of_the_main_policy():
    """what PAPER.md:104-106 fixes without any tie rule: whole blocks move, everyone ends inside the window, nothing is lost"""
    import numpy as np
    from paper_2006_00561_b200 import binding
    rng = np.random.default_rng(21)
    for world, B, maxexc in [(2, 1024, 1), (8, 1024, 1), (8, 1024, 2), (5, 1, 1), (16, 256, 3), (148, 1024, 1)]:
        for trial in range(20):
            T = rng.gamma(2.0, rng.choice([2000, 20480, 90000]) / 2.0, world).astype(np.int64)
            T[0] += 1
            ns, base, counts = binding.exchange_plan(T, binding.PA_POLICY_MAIN, B, maxexc)
            cnt, tot = np.diff(ns), int(T.sum())
            r = tot // world + (np.arange(world) < tot % world)
            assert cnt.sum() == tot and np.all(cnt >= 0)
            assert np.all((cnt - T) % B == 0)                         # blocks of B replicas
            assert np.all(np.abs(cnt - r) <= maxexc * B)              # the window `maxexc`
            inside = np.all(np.abs(T - r) <= maxexc * B)
            assert (not inside) or np.array_equal(cnt, T)             # nobody outside the window: nothing moves


def test_plan_check_gives_every_rank_the_same_verdict():
    """pa_dist_plan_check judges EVERY rank's share against THAT rank's capacity, so the rank that would overflow and the
    ranks that would not all refuse the step before anything is exchanged (a refusal on one rank only would leave the
    others waiting in the point-to-point exchange)"""
    import numpy as np
    from paper_2006_00561_b200 import binding
    # policy main moves whole blocks: r = 1000 each, born = (2100, 0, 900), B = 1024: e = (1100,-1000,-100) -> 0->1: (76,24,-100)
    ns, _, _ = binding.exchange_plan([2100, 0, 900], binding.PA_POLICY_MAIN, 1024, 1)
    assert np.diff(ns).tolist() == [1076, 1024, 900]
    binding.plan_check(ns, [1100, 1100, 1100])
    binding.plan_check(ns, None)
    with pytest.raises(binding.PaError) as e:
        binding.plan_check(ns, [1100, 1023, 1100])    # rank 1 alone cannot hold its share: every rank learns that
    assert e.value.code == binding.PA_ECAPACITY
    # an empty share (policy none, a rank without offspring; or fewer children than ranks)
    ns, _, _ = binding.exchange_plan([3000, 0, 500], binding.PA_POLICY_NONE)
    with pytest.raises(binding.PaError) as e:
        binding.plan_check(ns, [4096] * 3)
    assert e.value.code == binding.PA_EEXTINCT
    ns, _, _ = binding.exchange_plan([1, 0, 1, 0], binding.PA_POLICY_BALANCED)
    with pytest.raises(binding.PaError) as e:
        binding.plan_check(ns, None)
    assert e.value.code == binding.PA_EEXTINCT
    with pytest.raises(binding.PaError) as e:        # both defects: capacity wins, on every rank alike
        binding.plan_check(binding.exchange_plan([3000, 0, 500], binding.PA_POLICY_NONE)[0], [100, 100, 100])
    assert e.value.code == binding.PA_ECAPACITY
    with pytest.raises(binding.PaError) as e:
        binding.plan_check([0, 1 << 31, (1 << 32) - 4096], None)   # global slot indices are 32-bit
    assert e.value.code == binding.PA_ECAPACITY


def _sharded_oracle_worker(rank, world, port, q, L, R0, seed, betas, theta, policy, glass_seed=None):
    """one rank of the partitioned run on the CPU: the oracle does the rank's arithmetic with GLOBAL replica indices as
    keys, the product's host plan (pa_dist_exchange_plan) and exchange (dist.exchange_slices over gloo) move the replicas"""
    os.environ.update({"RANK": str(rank), "WORLD_SIZE": str(world), "LOCAL_RANK": str(rank),
                       "MASTER_ADDR": "127.0.0.1", "MASTER_PORT": str(port)})
    import numpy as np
    import torch
    from paper_2006_00561_b200 import binding, dist
    from oracle import pa_oracle as orc
    g = dist.init_from_env(backend="gloo", device_kind="cpu")
    orc.set_threads(1)
    wpr = orc.words_per_replica(L)
    from paper_2006_00561_b200 import inputs
    bonds = None if glass_seed is None else inputs.bond_sample(L, glass_seed)  # second Hamiltonian: every rank, same sample
    start = [r * (R0 // world) + min(r, R0 % world) for r in range(world + 1)]
    spins = orc.init_population(L, R0, seed)[start[rank]:start[rank + 1]].copy()  # keyed by the global replica index
    first, beta, sum_lnQ = start[rank], 0.0, 0.0
    for step, beta_next in enumerate(betas, 1):
        E, M = orc.energy_mag(L, spins, bonds)
        R_loc, dbeta = spins.shape[0], beta_next - beta
        w_sum = float(np.sum(np.exp(-dbeta * E.astype(np.float64))))  # the rank's sum of weights
        rows = dist.all_gather_doubles(g, [w_sum, float(R_loc)])
        sumw, R = 0.0, 0
        for r in rows:  # rank order
            sumw += r[0]
            R += int(r[1])
        Q = sumw / R
        tau = orc.tau_weights(E, dbeta, Q)
        tau_global = np.zeros(first + R_loc, np.float64)  # the sampler keys parent j by its GLOBAL index
        tau_global[first:] = tau
        n = orc.poisson_counts(tau_global, float(R0) / float(R), seed, step)[first:]
        off, T_loc = orc.exclusive_scan(n)
        children, _, _ = orc.copy_population(L, n, off, spins, E, M, T_loc)
        T_all = [int(r[0]) for r in dist.all_gather_doubles(g, [float(T_loc)])]
        ns, base, counts = binding.exchange_plan(T_all, policy, 16, 1)
        binding.plan_check(ns, [4 * R0] * world)
        new_n = int(ns[rank + 1] - ns[rank])
        send = torch.from_numpy(children.reshape(-1).view(np.uint8).copy())
        recv = torch.zeros(new_n * wpr * 4, dtype=torch.uint8)
        dist.exchange_slices(g, send, recv, counts, wpr * 4)
        spins = recv.numpy().view(np.uint32).reshape(new_n, wpr).copy()
        first = int(ns[rank])
        if theta > 0:
            T4, T8 = orc.thresholds(beta_next)
            orc.sweeps_slots(L, np.arange(first, first + new_n, dtype=np.uint32), spins, seed, step, theta, T4, T8,
                             bonds=bonds)
        beta = beta_next
        sum_lnQ += float(np.log(Q))
    q.put((rank, first, spins, sum_lnQ))
    dist.barrier(g)
    dist.shutdown(g)


@pytest.mark.parametrize("world,policy,glass_seed", [(2, 0, None), (4, 0, None), (3, 1, None), (2, 2, None), (2, 3, None),
                                                     (2, 0, 5), (3, 1, 6)])
def test_sharded_run_equals_the_single_population_run_gloo(world, policy, glass_seed):
    """world-size 2/3/4 over gloo: the concatenation of the ranks' populations equals the one-population oracle run bit
    for bit (random numbers are keyed by global replica index and global step; the policy only moves rank boundaries)"""
    import numpy as np
    from oracle import pa_oracle as orc
    L, R0, seed, theta = 8, 600, 77, 2
    betas = [0.05 * k for k in range(1, 9)]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_sharded_oracle_worker, args=(r, world, port, q, L, R0, seed, betas, theta, policy, glass_seed))
             for r in range(world)]
    for p in procs:
        p.start()
    res = sorted((q.get(timeout=300) for _ in procs), key=lambda t: t[0])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    from paper_2006_00561_b200 import inputs
    ref = orc.OraclePA(L, R0, seed=seed, bonds=None if glass_seed is None else inputs.bond_sample(L, glass_seed))
    for b in betas:
        ref.step(b, theta)
    got = np.concatenate([r[2] for r in res], axis=0)
    assert got.shape == ref.spins.shape and np.array_equal(got, ref.spins)
    assert [r[1] for r in res] == sorted(r[1] for r in res) and res[0][1] == 0   # ranks own increasing global ranges
    for r in res:
        assert abs(r[3] - ref.sum_lnQ) <= 1e-12 * abs(ref.sum_lnQ)               # same ln Z on every rank (rounding of Q only)
