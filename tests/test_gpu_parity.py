"""GPU parity: the CUDA path (through the C ABI, libsw.so) against the CPU oracle, bit for bit.

Bar (BASELINE.json north_star): identical spin configurations after every compared sweep, identical integer
bond/state histograms, identical canonical labels; derived doubles within 1e-12 relative (they are computed from
identical integers in a fixed order, so they are in fact identical).
"""
from __future__ import annotations

import math
from concurrent.futures import ThreadPoolExecutor

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

POTTS, CLOCK = 0, 1
GENERIC, TILED, SMALL, HAWICK, KALENTEV = 1, 2, 3, 4, 5


@pytest.fixture(scope="module")
def sw():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1202_0635_b200 import build, binding
    build.build()
    binding.load()
    return binding


def tc(q):
    return 1.0 / math.log(1.0 + math.sqrt(float(q)))


def _assert_same(a, b, what):
    if not np.array_equal(a, b):
        bad = np.argwhere(np.asarray(a) != np.asarray(b))
        raise AssertionError(f"{what}: {len(bad)} mismatches, first at {bad[:5].tolist()}")


def run_and_compare(sw, oracle, L, q, model, T, seed, algo, n, start=None, t0=0, labels=True, bonds=True):
    """n consecutive sweeps, everything compared after every sweep."""
    with sw.Lattice(L, q, model, T, seed, algo=algo) as lat:
        assert lat.algorithm == algo
        _assert_same(lat.get_thresholds(), oracle.thresholds(q, model, T), "thresholds")
        if start is None:
            s = oracle.init_spins(L, q, seed)
            _assert_same(lat.get_spins(), s, "initial spins")
        else:
            s = np.array(start, dtype=np.uint8).reshape(L, L)
            lat.set_spins(s, t0)
            _assert_same(lat.get_spins(), s, "set/get round trip")
        assert lat.sweep_index == t0
        for t in range(t0, t0 + n):
            if bonds:
                _assert_same(lat.debug_bonds(), oracle.bonds(L, q, model, T, seed, t, s), f"bonds of sweep {t}")
            bh, sh = lat.observables()
            obh, osh = oracle.observables(L, q, s)
            _assert_same(bh, obh, f"bond_hist before sweep {t}")
            _assert_same(sh, osh, f"state_hist before sweep {t}")
            lat.sweep(1)
            s, olab = oracle.sweep(L, q, model, T, seed, t, s, want_labels=True)
            if labels:
                _assert_same(lat.get_labels(), olab, f"labels of sweep {t}")
            _assert_same(lat.get_spins(), s, f"spins after sweep {t}")
        assert lat.sweep_index == t0 + n
        assert lat.launch_count > 0
    return s


# ------------------------------------------------------------------------------------------------
# generic back-end: any L >= 2 (odd sizes, the 2x2 multigraph, ragged last pair)
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("L", [2, 3, 5, 8, 31, 64, 100, 130])
@pytest.mark.parametrize("q,model,T", [(2, POTTS, tc(2)), (3, POTTS, tc(3)), (6, CLOCK, 0.9), (5, CLOCK, 0.7)])
def test_generic_small(sw, oracle, L, q, model, T):
    run_and_compare(sw, oracle, L, q, model, T, seed=0x5EED0001 + L, algo=GENERIC, n=6 if L <= 64 else 3)


def test_generic_high_seed_and_extreme_temperatures(sw, oracle):
    run_and_compare(sw, oracle, 48, 2, POTTS, tc(2), seed=(1 << 63) + 12345, algo=GENERIC, n=4)
    run_and_compare(sw, oracle, 48, 2, POTTS, 0.02, seed=7, algo=GENERIC, n=3)     # p -> 1 (threshold clamp), one cluster per domain
    run_and_compare(sw, oracle, 48, 4, POTTS, 1e6, seed=7, algo=GENERIC, n=3)      # p -> 0, every site a cluster
    run_and_compare(sw, oracle, 48, 16, POTTS, tc(16), seed=9, algo=GENERIC, n=3)  # q = SW_MAX_Q
    run_and_compare(sw, oracle, 48, 16, CLOCK, 0.5, seed=9, algo=GENERIC, n=3)


# ------------------------------------------------------------------------------------------------
# tiled back-end: several tiles in both directions, structured inputs, both models
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("L", [128, 256, 384])
@pytest.mark.parametrize("q,model,T", [(2, POTTS, tc(2)), (3, POTTS, tc(3)), (4, POTTS, tc(4)), (6, CLOCK, 0.9), (3, CLOCK, 0.6)])
def test_tiled_small(sw, oracle, L, q, model, T):
    run_and_compare(sw, oracle, L, q, model, T, seed=0x5EED0100 + L + q, algo=TILED, n=4 if L <= 256 else 2)


@pytest.mark.parametrize("q,model,T", [(2, POTTS, 0.02), (2, POTTS, 0.8 * tc(2)), (2, POTTS, 1e6), (6, CLOCK, 0.05), (16, POTTS, tc(16))])
def test_tiled_structured_inputs(sw, oracle, q, model, T):
    """Uniform lattice at low T (one cluster spanning every tile and both seams), stripes, checkerboard, domains."""
    from paper_1202_0635_b200 import workloads as w
    L = 256
    starts = [w.uniform_spins(L, q - 1), w.stripes(L, q, 5, True), w.stripes(L, q, 37, False), w.checkerboard(L, q),
              w.domains(L, q, 3, 48), w.random_spins(L, q, 4)]
    for k, st in enumerate(starts):
        run_and_compare(sw, oracle, L, q, model, T, seed=1000 + k, algo=TILED, n=2, start=st, t0=17 * k)


def test_tiled_equals_generic_on_device(sw):
    """Many sweeps without the oracle: both back-ends must stay identical (cheap hash of the whole run)."""
    L, q, T, seed = 512, 2, tc(2), 31337
    with sw.Lattice(L, q, POTTS, T, seed, algo=TILED) as a, sw.Lattice(L, q, POTTS, T, seed, algo=GENERIC) as b:
        for _ in range(10):
            a.sweep(20)
            b.sweep(20)
            assert np.array_equal(a.get_spins(), b.get_spins())
            assert np.array_equal(a.get_labels(), b.get_labels())


@pytest.mark.parametrize("L,q,model,T,n", [(1024, 2, POTTS, tc(2), 6000), (512, 6, CLOCK, 0.9, 6000), (1024, 2, POTTS, 0.8 * tc(2), 4000)])
def test_soak_tiled_graph_path_equals_generic(sw, L, q, model, T, n):
    """Thousands of sweeps through the CUDA-graph replay of the tiled back-end against the generic back-end (races in the
    shared-memory union-find or in the seam merge would show up as a diverging trajectory sooner or later)."""
    with sw.Lattice(L, q, model, T, 4242, algo=TILED) as a, sw.Lattice(L, q, model, T, 4242, algo=GENERIC) as b:
        for k in range(n // 1000):
            a.sweep(1000)
            b.sweep(1000)
            assert np.array_equal(a.get_spins(), b.get_spins()), k
        assert np.array_equal(a.get_labels(), b.get_labels())
        assert a.stats()[7] > 0


@pytest.mark.parametrize("L,q,model,T", [(256, 2, POTTS, tc(2)), (384, 6, CLOCK, 0.9)])
def test_graph_replay_equals_plain_launches_and_the_oracle(sw, oracle, L, q, model, T):
    """sw_sweep(n >= 16) of the tiled back-end replays chunks of 16 sweeps from a CUDA graph whose kernel nodes get their sweep
    index set before every replay; the result must equal sweep-by-sweep plain launches (labels included), also after
    an odd number of plain sweeps (other ping-pong parity) and after sw_set_spins moved the sweep index, and the oracle."""
    seed = 77
    with sw.Lattice(L, q, model, T, seed, algo=TILED) as a, sw.Lattice(L, q, model, T, seed, algo=TILED) as b:
        a.sweep(53)                                   # 3 chunks through the graph + 5 plain
        for _ in range(53):
            b.sweep(1)                                # plain launches only
        assert a.stats()[7] == 3 and b.stats()[7] == 0, "the graph path was not taken"
        assert np.array_equal(a.get_spins(), b.get_spins())
        assert np.array_equal(a.get_labels(), b.get_labels())
        s = oracle.run(L, q, model, T, seed, 0, 53, oracle.init_spins(L, q, seed))
        assert np.array_equal(a.get_spins(), s)
        a.sweep(1)
        a.sweep(32)                                   # other parity of the ping-pong: second graph
        s = oracle.run(L, q, model, T, seed, 53, 33, s)
        assert np.array_equal(a.get_spins(), s)
        a.set_spins(s, 1000)                          # the sweep index jumps
        a.sweep(16)
        s = oracle.run(L, q, model, T, seed, 1000, 16, s)
        assert np.array_equal(a.get_spins(), s)


# ------------------------------------------------------------------------------------------------
# API behaviour
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("algo,L", [(GENERIC, 64), (TILED, 256)])
def test_composition_resume_and_record(sw, oracle, algo, L):
    q, T, seed = 3, tc(3), 5
    with sw.Lattice(L, q, POTTS, T, seed, algo=algo) as a, sw.Lattice(L, q, POTTS, T, seed, algo=algo) as b:
        a.sweep(7)
        b.sweep(3)
        b.sweep(0)
        b.sweep_async(4)
        b.sync()
        assert np.array_equal(a.get_spins(), b.get_spins()) and a.sweep_index == b.sweep_index == 7
        # resume from a snapshot in a fresh context
        with sw.Lattice(L, q, POTTS, T, seed, algo=algo) as c:
            c.set_spins(a.get_spins(), 7)
            c.sweep(5)
            a.sweep(5)
            assert np.array_equal(a.get_spins(), c.get_spins())
        # record: row k = observables before the k-th sweep of the call
        s = a.get_spins()
        bh, sh = a.sweep_record(6)
        s_or, obh, osh = oracle.run(L, q, POTTS, T, seed, 12, 6, s, record=True)
        _assert_same(bh, obh, "recorded bond_hist")
        _assert_same(sh, osh, "recorded state_hist")
        _assert_same(a.get_spins(), s_or, "spins after sweep_record")
        assert a.sweep_index == 18
        # derived doubles (R11): the library's sw_derive_* on the GPU's integers against the ORACLE's own functions on
        # the oracle's integers, 1e-12 relative (north_star)
        for k in range(6):
            e_gpu, e_or = sw.potts_energy(L, bh[k]), oracle.potts_energy(L, obh[k])
            m_gpu, m_or = sw.potts_m2(q, sh[k]), oracle.potts_m2(q, osh[k])
            assert abs(e_gpu - e_or) <= 1e-12 * abs(e_or) and abs(m_gpu - m_or) <= 1e-12 * max(1.0, abs(m_or))
        u_gpu, u_or = sw.moment_ratio(q, sh), oracle.moment_ratio(q, osh)
        assert abs(u_gpu - u_or) <= 1e-12 * abs(u_or) and u_or >= 1.0


def test_set_spins_rejects_bad_values_and_errors(sw):
    with sw.Lattice(64, 3, POTTS, 1.0, 1) as lat:
        before = lat.get_spins()
        bad = before.copy()
        bad[5, 7] = 3
        with pytest.raises(sw.SwError):
            lat.set_spins(bad, 4)
        assert np.array_equal(lat.get_spins(), before) and lat.sweep_index == 0
        with pytest.raises(sw.SwError):
            lat.sweep(-1)
        with pytest.raises(sw.SwError):
            lat.get_labels()                     # no sweep executed yet
        with pytest.raises(sw.SwError):
            lat.set_algorithm(TILED)             # L = 64 is not a multiple of 128
    with pytest.raises(sw.SwError):
        sw.Lattice(64, 3, 7, 1.0, 1)
    with sw.Lattice(128, 2, POTTS, 1.0, 1, torch_memory=False) as lat:   # library-owned memory and stream
        lat.sweep(2)
        assert lat.get_spins().max() < 2


def test_clock_record_and_observables(sw, oracle):
    L, q, T, seed = 128, 6, 0.9, 77
    with sw.Lattice(L, q, CLOCK, T, seed) as lat:
        s0 = lat.get_spins()
        bh, sh = lat.sweep_record(5)
        s_or, obh, osh = oracle.run(L, q, CLOCK, T, seed, 0, 5, s0, record=True)
        _assert_same(bh, obh, "clock bond_hist")
        _assert_same(sh, osh, "clock state_hist")
        _assert_same(lat.get_spins(), s_or, "clock spins")
        for k in range(5):
            a, b = sw.clock_energy(q, bh[k]), oracle.clock_energy(q, obh[k])
            assert abs(a - b) <= 1e-12 * abs(b)
            assert abs(sw.clock_m(q, sh[k]) - oracle.clock_m(q, osh[k])) <= 1e-12 * L * L


# ------------------------------------------------------------------------------------------------
# NEXT-2: the one-CTA back-end (L <= 128, all sweeps of a call in one launch) and batches of lattices
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("L", [2, 3, 5, 8, 31, 64, 100, 128])
@pytest.mark.parametrize("q,model,T", [(2, POTTS, tc(2)), (3, POTTS, tc(3)), (6, CLOCK, 0.9), (16, CLOCK, 0.5)])
def test_small_backend(sw, oracle, L, q, model, T):
    seed = 0x5EED0100 + L
    run_and_compare(sw, oracle, L, q, model, T, seed=seed, algo=SMALL, n=4 if L <= 64 else 2)
    # n sweeps inside ONE launch, then the labels of the last one
    with sw.Lattice(L, q, model, T, seed) as lat:
        assert lat.algorithm == (SMALL if L <= 64 else TILED if L % 128 == 0 else GENERIC)   # what SW_ALGO_AUTO picks
        lat.set_algorithm(SMALL)
        before = lat.launch_count
        lat.sweep(9)
        assert lat.launch_count == before + 1 and lat.sweep_index == 9
        s = oracle.run(L, q, model, T, seed, 0, 8, oracle.init_spins(L, q, seed))
        s, olab = oracle.sweep(L, q, model, T, seed, 8, s, want_labels=True)
        _assert_same(lat.get_spins(), s, "spins after 9 sweeps in one launch")
        _assert_same(lat.get_labels(), olab, "labels of the last sweep")


@pytest.mark.parametrize("L,q,model", [(64, 2, POTTS), (32, 3, POTTS), (48, 6, CLOCK), (128, 2, POTTS), (7, 4, CLOCK),
                                       (256, 2, POTTS), (384, 3, POTTS), (256, 6, CLOCK)])
def test_batch_every_lattice_equals_its_own_run(sw, oracle, L, q, model):
    """A batch of lattices with different temperatures and seeds: lattice b equals the single-lattice oracle run with
    (T[b], seed[b]) after every call, and its histograms equal the oracle's.  L <= 128: one CTA per lattice; L = 256, 384:
    the tiles of all lattices in one grid per kernel."""
    B = 11 if L <= 128 else 5
    base = tc(q) if model == POTTS else 0.9
    T = [base * (0.6 + 0.08 * b) for b in range(B)]
    seed = [0x5EED0200 + 7919 * b + (b << 40) for b in range(B)]
    with sw.Batch(L, q, model, T, seed) as bt:
        want = [oracle.init_spins(L, q, seed[b]) for b in range(B)]
        got = bt.get_spins()
        for b in range(B):
            _assert_same(got[b], want[b], f"S^0 of lattice {b}")
        t = 0
        for n in (1, 6, 3):
            bt.sweep(n)
            got = bt.get_spins()
            for b in range(B):
                want[b] = oracle.run(L, q, model, T[b], seed[b], t, n, want[b])
                _assert_same(got[b], want[b], f"lattice {b} after sweep {t + n}")
            t += n
        assert bt.sweep_index == t
        bh, sh = bt.observables()
        for b in range(B):
            obh, osh = oracle.observables(L, q, want[b])
            _assert_same(bh[b], obh, f"bond_hist of lattice {b}")
            _assert_same(sh[b], osh, f"state_hist of lattice {b}")
        # hand-off: a configuration set from the host, absolute sweep index
        from paper_1202_0635_b200.workloads import random_spins
        s0 = np.stack([random_spins(L, q, 100 + b) for b in range(B)])
        bt.set_spins(s0, 40)
        bt.sweep(2)
        got = bt.get_spins()
        for b in range(B):
            _assert_same(got[b], oracle.run(L, q, model, T[b], seed[b], 40, 2, s0[b]), f"lattice {b} after the hand-off")


# ------------------------------------------------------------------------------------------------
# NEXT-4: the paper's own labellers as A/B back-ends, with their iteration counts
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("algo", [HAWICK, KALENTEV])
@pytest.mark.parametrize("L,q,model,T", [(2, 2, POTTS, tc(2)), (5, 3, POTTS, tc(3)), (31, 6, CLOCK, 0.9), (64, 2, POTTS, tc(2)),
                                          (128, 2, POTTS, 0.8 * tc(2)), (256, 2, POTTS, tc(2)), (100, 4, POTTS, 1e6), (48, 2, POTTS, 0.02)])
def test_paper_labellers_reach_the_oracle_labels(sw, oracle, algo, L, q, model, T):
    """Converged label equivalence = smallest site index of the cluster: labels, spins and histograms equal
    the oracle's after every sweep."""
    run_and_compare(sw, oracle, L, q, model, T, seed=0x5EED0400 + L, algo=algo, n=3)


@pytest.mark.parametrize("algo", [HAWICK, KALENTEV])
def test_paper_labellers_iteration_counts(sw, algo):
    """PAPER.md:75 quotes 6.6 / 7.1 iterations per sweep at Tc for L = 256 / 512 (q = 2).  The count depends on details the
    paper does not give (scan order, what counts as an iteration), so only the scale and the slow growth with L are
    checked: a handful of whole-lattice passes, more at L = 512 than at L = 256, one pass when nothing is bonded."""
    its = {}
    for L in (256, 512):
        with sw.Lattice(L, 2, POTTS, tc(2), 0x5EED0401, algo=algo) as lat:
            lat.sweep(60)                               # equilibrate: the cluster structure sets the count
            st0 = lat.stats()
            lat.sweep(40)
            st1 = lat.stats()
            its[L] = (st1[5] - st0[5]) / (st1[6] - st0[6])
            print(f"algo {algo} L={L}: {its[L]:.2f} iterations per sweep at Tc (paper: {6.6 if L == 256 else 7.1})")
    assert 3.0 <= its[256] <= 20.0 and 3.0 <= its[512] <= 20.0 and its[512] >= its[256] - 0.5
    with sw.Lattice(64, 2, POTTS, 1e6, 1, algo=algo) as lat:    # p -> 0: no bond, the first scan changes nothing
        lat.sweep(3)
        st = lat.stats()
        assert st[5] == 3 and st[6] == 3


# ------------------------------------------------------------------------------------------------
# BASELINE.json configs at full size
# ------------------------------------------------------------------------------------------------
def test_config1_L64_every_one_of_1000_sweeps(sw, oracle):
    from paper_1202_0635_b200.workloads import CONFIGS
    w = CONFIGS["c1_potts2_L64"]
    with sw.Lattice(w.L, w.q, w.model, w.T, w.seed) as lat:
        s = oracle.init_spins(w.L, w.q, w.seed)
        for t in range(w.sweeps):
            lat.sweep(1)
            s = oracle.sweep(w.L, w.q, w.model, w.T, w.seed, t, s)
            if t % 10 == 9 or t < 20:
                _assert_same(lat.get_spins(), s, f"config 1 spins after sweep {t}")
        _assert_same(lat.get_spins(), s, "config 1 final spins")
        bh, sh = lat.observables()
        obh, osh = oracle.observables(w.L, w.q, s)
        assert np.array_equal(bh, obh) and np.array_equal(sh, osh)


def _largest_cluster_fraction(labels):
    lab = np.asarray(labels).ravel()
    return float(np.bincount(lab).max()) / lab.size


def _snapshot_check(sw, oracle, w, early, lates, regime=None):
    """Sweeps 0..early-1 compared one by one; then, for every (t_at, n) of `lates`, the GPU runs alone to sweep t_at
    and n further sweeps are compared starting from GPU snapshots handed to the oracle (spins, t) -- SURVEY 8(c) row
    "GPU vs oracle".  Oracle sweeps run in parallel threads: each one starts from a GPU snapshot, so they are independent
    checks.  `regime` = (t, lo, hi): the largest-cluster fraction of the oracle's labels of sweep t (one of the compared
    sweeps) must lie in [lo, hi], so that a reader sees which cluster structure the snapshot exercised."""
    jobs = []  # (t, spins_before, spins_after_gpu, obs_before_gpu)
    with sw.Lattice(w.L, w.q, w.model, w.T, w.seed) as lat:
        assert lat.algorithm == TILED
        _assert_same(lat.get_thresholds(), oracle.thresholds(w.q, w.model, w.T), "thresholds")
        s_before = lat.get_spins()
        _assert_same(s_before, oracle.init_spins(w.L, w.q, w.seed), "initial spins")
        t_now = 0
        for t_at, n in [(0, early)] + list(lates):
            if n == 0:
                continue
            if t_at > t_now:
                lat.sweep(t_at - t_now)
                s_before = lat.get_spins()
            assert lat.sweep_index == t_at
            for t in range(t_at, t_at + n):
                obs = lat.observables()
                lat.sweep(1)
                s_after = lat.get_spins()
                jobs.append((t, s_before, s_after, obs))
                s_before = s_after
            t_now = t_at + n

    fractions = {}

    def check(job):
        t, sb, sa, (bh, sh) = job
        if regime is not None and t == regime[0]:
            want, lab = oracle.sweep(w.L, w.q, w.model, w.T, w.seed, t, sb, want_labels=True)
            fractions[t] = _largest_cluster_fraction(lab)
        else:
            want = oracle.sweep(w.L, w.q, w.model, w.T, w.seed, t, sb)
        obh, osh = oracle.observables(w.L, w.q, sb)
        return t, np.array_equal(want, sa), np.array_equal(bh, obh) and np.array_equal(sh, osh)

    with ThreadPoolExecutor(max_workers=8) as ex:
        for t, ok_s, ok_o in ex.map(check, jobs):
            assert ok_s, f"{w.name}: spins after sweep {t} differ from the oracle"
            assert ok_o, f"{w.name}: observables before sweep {t} differ from the oracle"
    if regime is not None:
        f = fractions[regime[0]]
        print(f"{w.name}: largest cluster of sweep {regime[0]} holds {f:.4f} of the sites")
        assert regime[1] <= f <= regime[2], f"{w.name}: largest-cluster fraction {f} outside [{regime[1]}, {regime[2]}] at sweep {regime[0]}"


def test_config2_L4096_potts2(sw, oracle):
    """sweeps 0..32 one by one, then snapshots at t = 1000, 6000, 10990 (the last sweeps of the config's
    1000 + 10000), a few sweeps each.  At Tc the largest cluster holds a sizeable fraction (L^(-1/8) scaling)."""
    from paper_1202_0635_b200.workloads import CONFIGS
    _snapshot_check(sw, oracle, CONFIGS["c2_potts2_L4096"], early=33, lates=[(1000, 3), (6000, 3), (10990, 3)], regime=(6001, 0.05, 0.8))


def test_config3_L4096_clock6(sw, oracle):
    from paper_1202_0635_b200.workloads import CONFIGS
    _snapshot_check(sw, oracle, CONFIGS["c3_clock6_L4096"], early=12, lates=[(1000, 2), (9990, 2)], regime=(1001, 0.0, 0.9))


def test_config4_L8192_potts3_and_4(sw, oracle):
    from paper_1202_0635_b200.workloads import CONFIGS
    _snapshot_check(sw, oracle, CONFIGS["c4_potts3_L8192"], early=3, lates=[(1000, 2)], regime=(1001, 0.0, 0.8))
    _snapshot_check(sw, oracle, CONFIGS["c4_potts4_L8192"], early=3, lates=[(1000, 2)], regime=(1001, 0.0, 0.8))


def test_config5_L16384_three_temperatures(sw, oracle):
    """Late snapshots matter: the spanning cluster at 0.8 Tc does not exist at t = 0.  At t = 300 it does (SURVEY 8(d):
    "one cluster holds 95 % of sites"); at 1.2 Tc the largest cluster is tiny."""
    from paper_1202_0635_b200.workloads import CONFIGS
    _snapshot_check(sw, oracle, CONFIGS["c5_potts2_L16384_0.8Tc"], early=1, lates=[(300, 2)], regime=(301, 0.85, 1.0))
    _snapshot_check(sw, oracle, CONFIGS["c5_potts2_L16384_Tc"], early=1, lates=[(300, 1)], regime=(300, 0.01, 0.8))
    _snapshot_check(sw, oracle, CONFIGS["c5_potts2_L16384_1.2Tc"], early=0, lates=[(300, 1)], regime=(300, 0.0, 0.01))


@pytest.mark.parametrize("L", [4096, 16384])
def test_full_size_structured_start_one_giant_root(sw, oracle, L):
    """A uniform lattice handed in at full size, cold (T = 0.02: every bond active, ONE cluster) and at 0.8 Tc (p = 0.67,
    a spanning cluster with holes): every tile's open roots funnel into one global root -- the worst case of the
    cross-tile union-find (2048 tiles at L = 4096, 32768 at L = 16384).  Spins AND canonical labels of two sweeps."""
    from paper_1202_0635_b200.workloads import uniform_spins
    q, seed, t0 = 2, 0x5EED0005, 5
    for T, lo in ((0.02, 0.999), (0.8 * tc(2), 0.85)):
        with sw.Lattice(L, q, POTTS, T, seed) as lat:
            assert lat.algorithm == TILED
            s = uniform_spins(L, 1)
            lat.set_spins(s, t0)
            for t in range(t0, t0 + 2):
                lat.sweep(1)
                s_gpu, lab_gpu = lat.get_spins(), lat.get_labels()
                s, olab = oracle.sweep(L, q, POTTS, T, seed, t, s, want_labels=True)
                _assert_same(lab_gpu, olab, f"L={L} T={T}: labels of sweep {t}")
                _assert_same(s_gpu, s, f"L={L} T={T}: spins after sweep {t}")
                if t == t0:
                    f = _largest_cluster_fraction(olab)
                    print(f"L={L} T={T:.4f}: largest cluster holds {f:.5f} of the sites")
                    assert f >= lo
                del lab_gpu, olab


# ------------------------------------------------------------------------------------------------
# NEXT-1: correlation histograms (eq.(5), (6); R15)
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("L,q,model,T", [(64, 6, CLOCK, 0.9), (130, 3, POTTS, tc(3)), (31, 5, CLOCK, 0.7), (256, 2, POTTS, tc(2))])
def test_correlation_matches_oracle(sw, oracle, L, q, model, T):
    seed = 0x5EED0C0D
    with sw.Lattice(L, q, model, T, seed) as lat:
        lat.sweep(3)
        s = lat.get_spins()
        for r in sorted({0, 1, 2, 3, L // 4, L // 2, L - 1}):
            _assert_same(lat.correlation(r), oracle.correlation(L, q, s, r), f"corr_hist r={r}")
        bh, _ = lat.observables()
        _assert_same(lat.correlation(1), bh, "corr_hist(1) == bond_hist")
        with pytest.raises(sw.SwError):
            lat.correlation(L)


def test_record_corr_rows_and_derived_doubles(sw, oracle):
    L, q, T, seed, n = 128, 6, 0.9, 0x5EED0C0E, 6
    with sw.Lattice(L, q, CLOCK, T, seed) as lat:
        bh, sh, c1, c2 = lat.sweep_record_corr(n, L // 4, L // 2)
    s = oracle.init_spins(L, q, seed)
    oq, oh = [], []
    for k in range(n):
        obh, osh = oracle.observables(L, q, s)
        _assert_same(bh[k], obh, f"bond row {k}")
        _assert_same(sh[k], osh, f"state row {k}")
        o1, o2 = oracle.correlation(L, q, s, L // 4), oracle.correlation(L, q, s, L // 2)
        _assert_same(c1[k], o1, f"corr(L/4) row {k}")
        _assert_same(c2[k], o2, f"corr(L/2) row {k}")
        oq.append(o1); oh.append(o2)
        g_gpu, g_or = sw.g(q, c1[k]), oracle.g(q, o1)             # eq.(5): library vs oracle, 1e-12 relative
        assert abs(g_gpu - g_or) <= 1e-12 * max(abs(g_or), 1e-300) and abs(g_gpu) <= 1.0
        s = oracle.sweep(L, q, CLOCK, T, seed, k, s)
    r_gpu, r_or = sw.ratio_R(q, c2, c1), oracle.ratio_R(q, np.array(oh), np.array(oq))   # eq.(6)
    assert abs(r_gpu - r_or) <= 1e-12 * abs(r_or)


def test_correlation_full_size_sampled(sw, oracle):
    """L=4096 clock lattice (config 3 shape): the full histogram at r = L/4 and L/2 against the oracle."""
    L, q, T, seed = 4096, 6, 0.9, 0x5EED0003
    with sw.Lattice(L, q, CLOCK, T, seed) as lat:
        lat.sweep(20)
        s = lat.get_spins()
        for r in (L // 4, L // 2, 5):
            _assert_same(lat.correlation(r), oracle.correlation(L, q, s, r), f"corr_hist r={r}")
