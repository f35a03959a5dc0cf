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
GENERIC, TILED = 1, 2


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
        # derived doubles (R11) from both sides' integers: within 1e-12 relative (identical in fact)
        for k in range(6):
            e_gpu, e_or = sw.potts_energy(L, bh[k]), sw.potts_energy(L, obh[k])
            m_gpu, m_or = sw.potts_m2(q, sh[k]), sw.potts_m2(q, osh[k])
            assert abs(e_gpu - e_or) <= 1e-12 * abs(e_or) and abs(m_gpu - m_or) <= 1e-12 * max(1.0, abs(m_or))


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
            a, b = sw.clock_energy(q, bh[k]), sw.clock_energy(q, obh[k])
            assert abs(a - b) <= 1e-12 * abs(b)
            assert abs(sw.clock_magnetisation(q, sh[k]) - sw.clock_magnetisation(q, osh[k])) <= 1e-12 * L * L


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


def _snapshot_check(sw, oracle, w, early, late_at, late):
    """Sweeps 0..early-1 compared one by one; then the GPU runs alone to sweep `late_at`, and `late` further sweeps
    are compared starting from GPU snapshots handed to the oracle (spins, t).  Oracle sweeps run in parallel threads:
    each one starts from a GPU snapshot, so they are independent checks."""
    jobs = []  # (t, spins_before, spins_after_gpu, obs_before_gpu)
    with sw.Lattice(w.L, w.q, w.model, w.T, w.seed) as lat:
        assert lat.algorithm == TILED
        _assert_same(lat.get_thresholds(), oracle.thresholds(w.q, w.model, w.T), "thresholds")
        s_before = lat.get_spins()
        _assert_same(s_before, oracle.init_spins(w.L, w.q, w.seed), "initial spins")
        for t in range(early):
            obs = lat.observables()
            lat.sweep(1)
            s_after = lat.get_spins()
            jobs.append((t, s_before, s_after, obs))
            s_before = s_after
        if late:
            lat.sweep(late_at - early)
            s_before = lat.get_spins()
            for t in range(late_at, late_at + late):
                obs = lat.observables()
                lat.sweep(1)
                s_after = lat.get_spins()
                jobs.append((t, s_before, s_after, obs))
                s_before = s_after

    def check(job):
        t, sb, sa, (bh, sh) = job
        want = oracle.sweep(w.L, w.q, w.model, w.T, w.seed, t, sb)
        obh, osh = oracle.observables(w.L, w.q, sb)
        return t, np.array_equal(want, sa), np.array_equal(bh, obh) and np.array_equal(sh, osh)

    with ThreadPoolExecutor(max_workers=8) as ex:
        for t, ok_s, ok_o in ex.map(check, jobs):
            assert ok_s, f"{w.name}: spins after sweep {t} differ from the oracle"
            assert ok_o, f"{w.name}: observables before sweep {t} differ from the oracle"


def test_config2_L4096_potts2(sw, oracle):
    from paper_1202_0635_b200.workloads import CONFIGS
    _snapshot_check(sw, oracle, CONFIGS["c2_potts2_L4096"], early=3, late_at=300, late=3)


def test_config3_L4096_clock6(sw, oracle):
    from paper_1202_0635_b200.workloads import CONFIGS
    _snapshot_check(sw, oracle, CONFIGS["c3_clock6_L4096"], early=2, late_at=200, late=2)


def test_config4_L8192_potts3_and_4(sw, oracle):
    from paper_1202_0635_b200.workloads import CONFIGS
    _snapshot_check(sw, oracle, CONFIGS["c4_potts3_L8192"], early=1, late_at=100, late=1)
    _snapshot_check(sw, oracle, CONFIGS["c4_potts4_L8192"], early=1, late_at=100, late=1)


def test_config5_L16384_three_temperatures(sw, oracle):
    """Late snapshots matter: the spanning cluster at 0.8 Tc does not exist at t = 0."""
    from paper_1202_0635_b200.workloads import CONFIGS
    _snapshot_check(sw, oracle, CONFIGS["c5_potts2_L16384_0.8Tc"], early=1, late_at=60, late=1)
    _snapshot_check(sw, oracle, CONFIGS["c5_potts2_L16384_Tc"], early=0, late_at=60, late=1)
    _snapshot_check(sw, oracle, CONFIGS["c5_potts2_L16384_1.2Tc"], early=0, late_at=60, late=1)


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
    for k in range(n):
        obh, osh = oracle.observables(L, q, s)
        _assert_same(bh[k], obh, f"bond row {k}")
        _assert_same(sh[k], osh, f"state row {k}")
        o1, o2 = oracle.correlation(L, q, s, L // 4), oracle.correlation(L, q, s, L // 2)
        _assert_same(c1[k], o1, f"corr(L/4) row {k}")
        _assert_same(c2[k], o2, f"corr(L/2) row {k}")
        g1, g2 = sw.correlation_g(q, c1[k]), sw.correlation_g(q, o1)
        assert g1 == g2 and abs(g1) <= 1.0
        s = oracle.sweep(L, q, CLOCK, T, seed, k, s)


def test_correlation_full_size_sampled(sw, oracle):
    """L=4096 clock lattice (config 3 shape): the full histogram at r = L/4 and L/2 against the oracle."""
    L, q, T, seed = 4096, 6, 0.9, 0x5EED0003
    with sw.Lattice(L, q, CLOCK, T, seed) as lat:
        lat.sweep(20)
        s = lat.get_spins()
        for r in (L // 4, L // 2, 5):
            _assert_same(lat.correlation(r), oracle.correlation(L, q, s, r), f"corr_hist r={r}")
