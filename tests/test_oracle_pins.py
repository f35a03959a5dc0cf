"""Pins of the CPU oracle against things other than itself (CPU only, ``-m "not gpu"``).

What each test fixes (DESIGN.md section 4 lists them beside the oracle function they pin):
  * Philox4x32-10            -> published known answers (tests/golden/philox4x32_10_kat.txt)
  * stream keying            -> DESIGN.md R5 table, word by word
  * thresholds               -> 60-digit mpmath evaluation of R1/R4/R6/R7 + SURVEY's printed integers
  * oracle_label             -> brute-force flood fill / exhaustive bond patterns on tiny tori
  * Potts sweep              -> exact Boltzmann distribution by enumeration (3x3, 4x4 tori), state level and
                                energy level; Kaufman's exact finite-torus Ising energy at L=64 (Onsager)
  * clock sweep              -> exact Boltzmann distribution of PAPER.md eq.(4) by enumeration (2x2 state level,
                                3x3 energy level, q = 2..6)
  * observables              -> direct numpy restatement with np.roll
"""
from __future__ import annotations

import itertools
import math
from collections import deque
from pathlib import Path

import mpmath
import numpy as np
import pytest

GOLD = Path(__file__).resolve().parent / "golden"
POTTS, CLOCK = 0, 1
TC2 = 1.0 / math.log(1.0 + math.sqrt(2.0))


def _gold_lines(name):
    for line in (GOLD / name).read_text().splitlines():
        line = line.strip()
        if line and not line.startswith("#"):
            yield line


# ------------------------------------------------------------------------------------------------
# Philox4x32-10 and the stream keying
# ------------------------------------------------------------------------------------------------
def test_philox_known_answers(oracle):
    n = 0
    for line in _gold_lines("philox4x32_10_kat.txt"):
        w = [int(x, 16) for x in line.replace("->", " ").split()]
        assert len(w) == 10
        got = oracle.philox4x32_10(w[0:4], w[4:6])
        assert [int(x) for x in got] == w[6:10], line
        n += 1
    assert n == 3


def _mulhi(w, q):
    return (int(w) * q) >> 32


@pytest.mark.parametrize("seed", [1, 0x5EED0002, (1 << 63) + 12345])
def test_stream_keying_matches_design_table(oracle, seed):
    """DESIGN.md R5: INIT (i>>2,0,3,0)[i&3]; AXIS (0,t,2,0)[0]; BOND (i>>1,t,0,0)[2(i&1)+d];
    CLUSTER (r>>2,t,1,0)[r&3]; key = (seed lo, seed hi)."""
    key = [seed & 0xFFFFFFFF, seed >> 32]
    L, q, t = 6, 5, 7
    N = L * L
    s0 = oracle.init_spins(L, q, seed).reshape(-1)
    for i in range(N):
        w = oracle.philox4x32_10([i >> 2, 0, 3, 0], key)[i & 3]
        assert s0[i] == _mulhi(w, q)
    for tt in (0, 1, 12345):
        assert oracle.axis(q, seed, tt) == _mulhi(oracle.philox4x32_10([0, tt, 2, 0], key)[0], q)
    # bonds: all spins equal => threshold is the Potts constant for every bond
    T = 1.3
    thr = oracle.potts_threshold(T)
    b = oracle.bonds(L, q, POTTS, T, seed, t, np.zeros((L, L), np.uint8)).reshape(-1)
    for i in range(N):
        ws = oracle.philox4x32_10([i >> 1, t, 0, 0], key)
        for d in (0, 1):
            assert ((b[i] >> d) & 1) == (1 if int(ws[2 * (i & 1) + d]) < thr else 0)
    # cluster decisions: arbitrary label array
    rng = np.random.default_rng(3)
    labels = rng.integers(0, N, size=(L, L), dtype=np.int32)
    out = oracle.flip(L, q, POTTS, seed, t, labels, np.zeros((L, L), np.uint8)).reshape(-1)
    for i, r in enumerate(labels.reshape(-1)):
        r = int(r)
        w = oracle.philox4x32_10([r >> 2, t, 1, 0], key)[r & 3]
        assert out[i] == _mulhi(w, q)
    # clock: flip iff top bit, reflection p -> (m - p) mod q
    m = oracle.axis(q, seed, t)
    sp = rng.integers(0, q, size=(L, L), dtype=np.uint8)
    out = oracle.flip(L, q, CLOCK, seed, t, labels, sp).reshape(-1)
    for i, r in enumerate(labels.reshape(-1)):
        r = int(r)
        w = int(oracle.philox4x32_10([r >> 2, t, 1, 0], key)[r & 3])
        want = (m - int(sp.reshape(-1)[i])) % q if (w >> 31) else int(sp.reshape(-1)[i])
        assert out[i] == want


# ------------------------------------------------------------------------------------------------
# Thresholds
# ------------------------------------------------------------------------------------------------
def _mp_thr(p):
    v = int(mpmath.floor(p * (mpmath.mpf(2) ** 32)))
    return max(0, min(v, 0xFFFFFFFF))


def test_potts_thresholds_high_precision_and_golden(oracle):
    mpmath.mp.dps = 60
    for line in _gold_lines("thresholds.txt"):
        f = line.split()
        if f[0] != "potts":
            continue
        q, fac, want = int(f[1]), float(f[2]), int(f[3])
        T = fac * (1.0 / math.log(1.0 + math.sqrt(float(q))))
        got = oracle.potts_threshold(T)
        assert got == want, line
        assert got == _mp_thr(1 - mpmath.exp(-1 / mpmath.mpf(T)))
    # closed form at the self-dual point: p_c = sqrt(q) / (1 + sqrt(q))  (PAPER.md:75 with eq.(1))
    for q in (2, 3, 4, 5, 7):
        T = 1.0 / math.log(1.0 + math.sqrt(float(q)))
        pc = mpmath.sqrt(q) / (1 + mpmath.sqrt(q))
        assert abs(oracle.potts_threshold(T) - _mp_thr(pc)) <= 1024  # T is a rounded double
    assert oracle.potts_threshold(1.0 / math.log(3.0)) == 0xAAAAAAAA  # q=4: p = 2/3
    # random temperatures, and the clamps of R7
    rng = np.random.default_rng(11)
    for T in rng.uniform(0.05, 20.0, size=200):
        assert abs(oracle.potts_threshold(float(T)) - _mp_thr(1 - mpmath.exp(-1 / mpmath.mpf(float(T))))) <= 1
    assert oracle.potts_threshold(1e-3) == 0xFFFFFFFF
    assert oracle.potts_threshold(1e300) == 0


def test_clock_table_high_precision_and_golden(oracle):
    mpmath.mp.dps = 60
    T = 0.9
    tab = oracle.clock_table(6, T)
    mag = {"h": mpmath.mpf(1) / 2, "r": mpmath.sqrt(3) / 2, "o": mpmath.mpf(1)}
    cls = {1: "h", 2: "r", 3: "o", 4: "r", 5: "h"}      # |sin(pi c / 6)| for c = 1..5
    golden = {}
    for line in _gold_lines("thresholds.txt"):
        f = line.split()
        if f[0] == "clock6":
            golden[(f[1], f[2])] = int(f[3])
            golden[(f[2], f[1])] = int(f[3])
    assert len(golden) == 9
    for ci in range(12):
        for cj in range(12):
            zero = (ci % 6 == 0) or (cj % 6 == 0) or ((ci < 6) != (cj < 6))
            if zero:
                assert tab[ci, cj] == 0
            else:
                a, b = cls[ci % 6], cls[cj % 6]
                assert tab[ci, cj] == golden[(a, b)]
                assert tab[ci, cj] == _mp_thr(1 - mpmath.exp(-2 * mag[a] * mag[b] / mpmath.mpf(T)))
    assert np.array_equal(tab, tab.T)
    # generic q, T: s(c) = sin(pi c / q) evaluated with 60 digits
    for q, T in ((2, 1.1), (3, 0.7), (4, 1.0), (5, 0.9), (8, 0.6)):
        tab = oracle.clock_table(q, T)
        for ci in range(2 * q):
            for cj in range(2 * q):
                si = mpmath.mpf(0) if ci % q == 0 else mpmath.sin(mpmath.pi * ci / q)
                sj = mpmath.mpf(0) if cj % q == 0 else mpmath.sin(mpmath.pi * cj / q)
                want = _mp_thr(1 - mpmath.exp(-2 * si * sj / mpmath.mpf(T))) if si * sj > 0 else 0
                assert abs(int(tab[ci, cj]) - want) <= 1, (q, T, ci, cj)


# ------------------------------------------------------------------------------------------------
# Cluster labeling against brute force
# ------------------------------------------------------------------------------------------------
def _bond_list(L):
    """(i, j) for every owned bond, ordered (site, direction) like the bit layout of bonds[]."""
    out = []
    for y in range(L):
        for x in range(L):
            i = y * L + x
            out.append((i, y * L + (x + 1) % L))
            out.append((i, ((y + 1) % L) * L + x))
    return out


def _flood_fill_labels(L, bonds):
    """Brute force: BFS from every site, label = min index reached."""
    N = L * L
    adj = [[] for _ in range(N)]
    flat = np.asarray(bonds).reshape(-1)
    for k, (i, j) in enumerate(_bond_list(L)):
        if (flat[i] >> (k & 1)) & 1:
            adj[i].append(j)
            adj[j].append(i)
    lab = np.zeros(N, dtype=np.int32)
    for s in range(N):
        seen = {s}
        dq = deque([s])
        while dq:
            u = dq.popleft()
            for v in adj[u]:
                if v not in seen:
                    seen.add(v)
                    dq.append(v)
        lab[s] = min(seen)
    return lab.reshape(L, L)


@pytest.mark.parametrize("L", [2, 3])
def test_label_exhaustive_bond_patterns(oracle, L):
    """Every one of the 2^(2N) bond patterns of the 2x2 (multigraph, R8) and 3x3 torus."""
    N = L * L
    bl = _bond_list(L)
    nb = len(bl)
    P = 1 << nb
    pat = np.arange(P, dtype=np.int64)
    lab = np.broadcast_to(np.arange(N, dtype=np.int32), (P, N)).copy()
    active = [((pat >> k) & 1).astype(bool) for k in range(nb)]
    for _ in range(N):                                   # min-propagation to the fixed point
        for k, (i, j) in enumerate(bl):
            m = np.minimum(lab[:, i], lab[:, j])
            lab[:, i] = np.where(active[k], m, lab[:, i])
            lab[:, j] = np.where(active[k], m, lab[:, j])
    step = 1 if L == 2 else 37                            # 3x3: every 37th pattern (7085 cases) + corners
    idx = list(range(0, P, step)) + [P - 1]
    for p in idx:
        bonds = np.zeros(N, dtype=np.uint8)
        for k, (i, _) in enumerate(bl):
            if (p >> k) & 1:
                bonds[i] |= 1 << (k & 1)
        got = oracle.label(L, bonds).reshape(-1)
        assert np.array_equal(got, lab[p]), (L, p)


@pytest.mark.parametrize("L,density,seed", [(4, 0.3, 0), (5, 0.5, 1), (7, 0.45, 2), (8, 0.6, 3), (8, 0.2, 4), (6, 1.0, 5), (6, 0.0, 6)])
def test_label_random_patterns_vs_flood_fill(oracle, L, density, seed):
    rng = np.random.default_rng(seed)
    for _ in range(20):
        bonds = (rng.random((L, L)) < density).astype(np.uint8) | ((rng.random((L, L)) < density).astype(np.uint8) << 1)
        assert np.array_equal(oracle.label(L, bonds), _flood_fill_labels(L, bonds))


def test_label_seam_cases(oracle):
    """A cluster that exists only through the periodic seam must take the min index across it."""
    L = 5
    bonds = np.zeros((L, L), np.uint8)
    bonds[2, L - 1] = 1                                   # (4,2) -+x-> (0,2): wraps in x
    bonds[L - 1, 3] |= 2                                  # (3,4) -+y-> (3,0): wraps in y
    lab = oracle.label(L, bonds)
    assert lab[2, L - 1] == 2 * L + 0 and lab[2, 0] == 2 * L + 0
    assert lab[L - 1, 3] == 3 and lab[0, 3] == 3
    assert np.array_equal(lab, _flood_fill_labels(L, bonds))
    # a ring around the torus in x on the last row, labelled by its first site
    bonds = np.zeros((L, L), np.uint8)
    bonds[L - 1, :] = 1
    lab = oracle.label(L, bonds)
    assert (lab[L - 1, :] == (L - 1) * L).all()
    assert (lab[: L - 1] == np.arange((L - 1) * L).reshape(L - 1, L)).all()


# ------------------------------------------------------------------------------------------------
# Observables
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("L,q", [(2, 2), (3, 3), (8, 6), (16, 4)])
def test_observables_vs_numpy_roll(oracle, L, q):
    rng = np.random.default_rng(L * 10 + q)
    s = rng.integers(0, q, size=(L, L), dtype=np.uint8)
    bh, sh = oracle.observables(L, q, s)
    si = s.astype(np.int64)
    d = np.concatenate([((si - np.roll(si, -1, axis=1)) % q).reshape(-1), ((si - np.roll(si, -1, axis=0)) % q).reshape(-1)])
    assert np.array_equal(bh, np.bincount(d, minlength=q))
    assert np.array_equal(sh, np.bincount(si.reshape(-1), minlength=q))
    assert bh.sum() == 2 * L * L and sh.sum() == L * L


# ------------------------------------------------------------------------------------------------
# Potts sweep = a valid SW update: exact enumeration of the Boltzmann distribution
# ------------------------------------------------------------------------------------------------
def _all_states(L, q):
    N = L * L
    n = q ** N
    idx = np.arange(n, dtype=np.int64)
    st = np.empty((n, N), dtype=np.int8)
    for k in range(N):
        st[:, k] = (idx // (q ** k)) % q
    return st


def _n_eq(st, L):
    n = np.zeros(st.shape[0], dtype=np.int64)
    for (i, j) in _bond_list(L):
        n += st[:, i] == st[:, j]
    return n


def _chi2(counts, expected):
    counts = np.asarray(counts, dtype=np.float64)
    expected = np.asarray(expected, dtype=np.float64)
    keep = expected > 0
    assert counts[~keep].sum() == 0
    return float((((counts - expected) ** 2)[keep] / expected[keep]).sum()), int(keep.sum()) - 1


def test_ising_density_of_states_golden():
    """The golden g(n_eq) rows are what brute force gives (so later tests may lean on them)."""
    for line in _gold_lines("ising_torus_dos.txt"):
        f = line.split()
        L = int(f[0])
        want = {int(a.split(":")[0]): int(a.split(":")[1]) for a in f[1:]}
        n = _n_eq(_all_states(L, 2), L)
        vals, cnt = np.unique(n, return_counts=True)
        assert dict(zip(vals.tolist(), cnt.tolist())) == want


@pytest.mark.parametrize("L,q,T,sweeps", [(3, 2, TC2, 120000), (4, 2, TC2, 120000), (3, 3, 0.9949728610718, 120000),
                                           (3, 4, 0.91, 80000), (3, 2, 0.7, 80000), (3, 2, 2.5, 80000)])
def test_potts_energy_histogram_is_boltzmann(oracle, L, q, T, sweeps):
    """Histogram of n_eq over a long oracle run vs sum_states delta(n_eq) exp(n_eq/T) / Z  (H = J(2N - n_eq))."""
    st = _all_states(L, q)
    n = _n_eq(st, L)
    w = np.exp((n - n.max()) / T)
    prob = np.bincount(n, weights=w, minlength=2 * L * L + 1)
    prob /= prob.sum()
    s0 = oracle.init_spins(L, q, 99)
    burn = 200
    _, bh, _ = oracle.run(L, q, POTTS, T, 99, 0, burn + sweeps, s0, record=True)
    neq = bh[burn::2, 0]                                   # thin by 2: SW on a 3x3 decorrelates in ~1 sweep
    counts = np.bincount(neq, minlength=2 * L * L + 1)
    mask = prob * len(neq) >= 5
    c = np.append(counts[mask], counts[~mask].sum())
    e = np.append(prob[mask], prob[~mask].sum()) * len(neq)
    chi2, dof = _chi2(c, e)
    assert chi2 < dof + 5.0 * math.sqrt(2.0 * dof) + 5, (chi2, dof)
    mean_exact = float((prob * np.arange(len(prob))).sum())
    err = float(neq.std() / math.sqrt(len(neq) / 3.0))
    assert abs(neq.mean() - mean_exact) < 5 * err, (neq.mean(), mean_exact, err)


@pytest.mark.parametrize("q,T", [(2, TC2), (3, 1.2)])
def test_potts_state_level_distribution_3x3(oracle, q, T):
    """Every one of the q^9 configurations is visited with its Boltzmann weight (catches errors that keep the
    energy histogram intact, e.g. a wrong wrap or a non-uniform new state)."""
    L = 3
    st = _all_states(L, q)
    n = _n_eq(st, L)
    prob = np.exp((n - n.max()) / T)
    prob /= prob.sum()
    powers = (q ** np.arange(L * L)).astype(np.int64)
    sweeps = 150000 if q == 2 else 300000
    s = oracle.init_spins(L, q, 5)
    counts = np.zeros(q ** (L * L), dtype=np.int64)
    for t in range(sweeps):
        s = oracle.sweep(L, q, POTTS, T, 5, t, s)
        if t >= 100 and (t & 1):
            counts[int((s.reshape(-1).astype(np.int64) * powers).sum())] += 1
    tot = counts.sum()
    mask = prob * tot >= 5
    c = np.append(counts[mask], counts[~mask].sum())
    e = np.append(prob[mask], prob[~mask].sum()) * tot
    chi2, dof = _chi2(c, e)
    assert chi2 < dof + 5.0 * math.sqrt(2.0 * dof), (chi2, dof)


# ------------------------------------------------------------------------------------------------
# Ising energy at large L: Kaufman's exact finite-torus partition function (-> Onsager as L -> inf)
# ------------------------------------------------------------------------------------------------
def _kaufman_logZ(n, K):
    """ln Z of the Ising model, weight exp(K sum sigma sigma), on an n x n torus (Kaufman 1949)."""
    K = mpmath.mpf(K)
    N = n * n

    def gamma(l):
        if l == 0:
            return 2 * K + mpmath.log(mpmath.tanh(K))
        return mpmath.acosh(mpmath.cosh(2 * K) * mpmath.coth(2 * K) - mpmath.cos(l * mpmath.pi / n))

    p1 = mpmath.mpf(1); p2 = mpmath.mpf(1); p3 = mpmath.mpf(1); p4 = mpmath.mpf(1)
    for r in range(n):
        go, ge = gamma(2 * r + 1), gamma(2 * r)
        p1 *= 2 * mpmath.cosh(n * go / 2)
        p2 *= 2 * mpmath.sinh(n * go / 2)
        p3 *= 2 * mpmath.cosh(n * ge / 2)
        p4 *= 2 * mpmath.sinh(n * ge / 2)
    return mpmath.log(mpmath.mpf(1) / 2) + (mpmath.mpf(N) / 2) * mpmath.log(2 * mpmath.sinh(2 * K)) + mpmath.log(p1 + p2 + p3 + p4)


def _kaufman_neq_density(n, T):
    """<n_eq> / 2N for eq.(1) at temperature T: n_eq = N + (sum sigma sigma)/2, K = 1/(2T)."""
    mpmath.mp.dps = 40
    N = n * n
    dlogZ = mpmath.diff(lambda k: _kaufman_logZ(n, k), mpmath.mpf(1) / (2 * mpmath.mpf(T)))
    return float((N + dlogZ / 2) / (2 * N))


def test_kaufman_formula_matches_brute_force_4x4():
    mpmath.mp.dps = 40
    for line in _gold_lines("ising_torus_dos.txt"):
        f = line.split()
        L = int(f[0])
        g = {int(a.split(":")[0]): int(a.split(":")[1]) for a in f[1:]}
        for K in (0.2, 0.4406867935, 0.8):
            Z = sum(c * mpmath.exp(mpmath.mpf(K) * (2 * n - 2 * L * L)) for n, c in g.items())
            assert abs(_kaufman_logZ(L, K) - mpmath.log(Z)) < mpmath.mpf(10) ** -25
        # and the energy it implies, against the two densities SURVEY.md section 8(c) prints
        want = {3: 0.9028116, 4: 0.8914059}[L]
        assert abs(_kaufman_neq_density(L, TC2) - want) < 2e-7


def test_kaufman_reaches_onsager():
    """Infinite-lattice value at Tc: <delta> per bond = (1 + 1/sqrt 2)/2 (Onsager); finite size adds ~0.1556/L."""
    ons = (1.0 + 1.0 / math.sqrt(2.0)) / 2.0
    assert abs(_kaufman_neq_density(64, TC2) - 0.8559846) < 2e-7
    assert abs(_kaufman_neq_density(256, TC2) - (ons + 0.1556 / 256)) < 2e-6


@pytest.mark.parametrize("fac,L", [(1.0, 64), (0.8, 48), (1.2, 48)])
def test_ising_energy_matches_kaufman(oracle, fac, L):
    T = fac * TC2
    exact = _kaufman_neq_density(L, T)
    s0 = oracle.init_spins(L, 2, 1234)
    burn, n = 300, 4000
    _, bh, sh = oracle.run(L, 2, POTTS, T, 1234, 0, burn + n, s0, record=True)
    x = bh[burn:, 0] / (2.0 * L * L)
    nb = 20                                                # batch means for the error bar
    bm = x[: (len(x) // nb) * nb].reshape(nb, -1).mean(axis=1)
    err = bm.std(ddof=1) / math.sqrt(nb)
    assert abs(x.mean() - exact) < 4.5 * err + 1e-5, (x.mean(), exact, err)
    assert err < 1.5e-3                                    # tight enough to tell 0.8560 (L=64) from Onsager's 0.8536
    assert (sh.sum(axis=1) == L * L).all() and (bh.sum(axis=1) == 2 * L * L).all()


@pytest.mark.parametrize("q", [3, 4])
def test_potts_self_dual_point_bond_density(oracle, q):
    """At Tc = 1/ln(1+sqrt q) the model is self-dual: <delta> -> (1+1/sqrt q)/2 and the active-bond
    density p_c <delta> -> 1/2 (finite-size corrections ~L^-0.8 (q=3), ~L^-0.5 (q=4))."""
    L = 48
    T = 1.0 / math.log(1.0 + math.sqrt(float(q)))
    s = oracle.init_spins(L, q, 77)
    dens = []
    for t in range(1500):
        s, b = oracle.sweep(L, q, POTTS, T, 77, t, s, want_bonds=True)
        if t >= 300:
            dens.append(((b & 1).sum() + (b >> 1).sum()) / (2.0 * L * L))
    assert abs(np.mean(dens) - 0.5) < 0.02, np.mean(dens)


# ------------------------------------------------------------------------------------------------
# Clock sweep (Wolff embedding, R4) = valid update of PAPER.md eq.(4): exact enumeration
# ------------------------------------------------------------------------------------------------
def _clock_energy2(st, L, q):
    """2 * sum over owned bonds of cos(2 pi (s_i - s_j)/q), rounded to 1e-9 units as int64 keys are not possible
    for general q -> returned as float64."""
    c = np.cos(2.0 * np.pi * np.arange(q) / q)
    e = np.zeros(st.shape[0], dtype=np.float64)
    for (i, j) in _bond_list(L):
        e += c[(st[:, i].astype(np.int64) - st[:, j]) % q]
    return e                                              # = -H/J


@pytest.mark.parametrize("q,T", [(6, 2.5), (6, 0.9), (5, 1.5), (4, 1.2), (3, 1.0), (2, 2.0)])
def test_clock_state_level_distribution_2x2(oracle, q, T):
    """2x2 torus (each site owns 2 bonds, so every pair is doubly bonded; R8): every configuration is visited
    with weight exp(-H/T), H from PAPER.md eq.(4)."""
    L = 2
    st = _all_states(L, q)
    mh = _clock_energy2(st, L, q)
    prob = np.exp((mh - mh.max()) / T)
    prob /= prob.sum()
    powers = (q ** np.arange(L * L)).astype(np.int64)
    sweeps = 250000
    s = oracle.init_spins(L, q, 21)
    counts = np.zeros(q ** (L * L), dtype=np.int64)
    for t in range(sweeps):
        s = oracle.sweep(L, q, CLOCK, T, 21, t, s)
        if t >= 100 and (t % 3 == 0):
            counts[int((s.reshape(-1).astype(np.int64) * powers).sum())] += 1
    tot = counts.sum()
    mask = prob * tot >= 5
    c = np.append(counts[mask], counts[~mask].sum())
    e = np.append(prob[mask], prob[~mask].sum()) * tot
    chi2, dof = _chi2(c, e)
    assert chi2 < dof + 5.0 * math.sqrt(2.0 * dof) + 5, (chi2, dof)


@pytest.mark.parametrize("q,T,sweeps", [(6, 0.9, 150000), (6, 0.7, 150000), (4, 1.0, 100000), (3, 0.8, 100000), (5, 1.0, 100000)])
def test_clock_energy_histogram_3x3(oracle, q, T, sweeps):
    L = 3
    st = _all_states(L, q)
    mh = _clock_energy2(st, L, q)
    key = np.rint(mh * 2.0 * 1e6).astype(np.int64)         # energies are multiples of small algebraic numbers
    levels, inv = np.unique(key, return_inverse=True)
    w = np.exp((mh - mh.max()) / T)
    prob = np.bincount(inv, weights=w, minlength=len(levels))
    prob /= prob.sum()
    c = np.cos(2.0 * np.pi * np.arange(q) / q)
    s0 = oracle.init_spins(L, q, 8)
    burn = 300
    _, bh, _ = oracle.run(L, q, CLOCK, T, 8, 0, burn + sweeps, s0, record=True)
    mh_run = (bh[burn::4].astype(np.float64) * c[None, :]).sum(axis=1)
    krun = np.rint(mh_run * 2.0 * 1e6).astype(np.int64)
    pos = np.searchsorted(levels, krun)
    assert (levels[pos] == krun).all()
    counts = np.bincount(pos, minlength=len(levels))
    tot = counts.sum()
    mask = prob * tot >= 5
    cc = np.append(counts[mask], counts[~mask].sum())
    ee = np.append(prob[mask], prob[~mask].sum()) * tot
    chi2, dof = _chi2(cc, ee)
    assert chi2 < dof + 5.0 * math.sqrt(2.0 * dof) + 5, (chi2, dof)
    mean_exact = float((prob * (levels / 2.0e6)).sum())
    err = float(mh_run.std() / math.sqrt(len(mh_run) / 3.0))
    assert abs(mh_run.mean() - mean_exact) < 5 * err, (mh_run.mean(), mean_exact, err)


# ------------------------------------------------------------------------------------------------
# Invariants of a sweep
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("q,model,T", [(2, POTTS, TC2), (3, POTTS, 0.995), (6, CLOCK, 0.9), (4, CLOCK, 0.8)])
def test_sweep_invariants(oracle, q, model, T):
    L, seed = 24, 4242
    s = oracle.init_spins(L, q, seed)
    assert s.max() < q
    for t in range(6):
        m = oracle.axis(q, seed, t)
        s2, lab, b = oracle.sweep(L, q, model, T, seed, t, s, want_labels=True, want_bonds=True)
        flat, lf = s.reshape(-1).astype(int), lab.reshape(-1)
        assert (lf <= np.arange(L * L)).all() and (lf[lf] == lf).all()
        assert np.array_equal(lab, _flood_fill_labels(L, b)) if t == 0 else True
        # bonds only between compatible spins
        right, down = np.roll(s, -1, axis=1), np.roll(s, -1, axis=0)
        if model == POTTS:
            assert ((b & 1) <= (s == right)).all() and ((b >> 1) <= (s == down)).all()
            for r in np.unique(lf):                       # every cluster uniform after the sweep
                assert len(np.unique(s2.reshape(-1)[lf == r])) == 1
        else:
            f2 = s2.reshape(-1).astype(int)
            for r in np.unique(lf):
                sel = lf == r
                assert (f2[sel] == flat[sel]).all() or (f2[sel] == (m - flat[sel]) % q).all()
        assert s2.max() < q
        s = s2


def test_sweep_composition_and_seeds(oracle):
    L, q, T = 16, 3, 0.995
    s0 = oracle.init_spins(L, q, 1)
    a = oracle.run(L, q, POTTS, T, 1, 0, 7, s0)
    b = oracle.run(L, q, POTTS, T, 1, 3, 4, oracle.run(L, q, POTTS, T, 1, 0, 3, s0))
    assert np.array_equal(a, b)
    assert np.array_equal(s0, oracle.init_spins(L, q, 1))
    assert not np.array_equal(s0, oracle.init_spins(L, q, 2))
    assert not np.array_equal(s0, oracle.init_spins(L, q, 1 + (1 << 32)))   # high key word is used
    assert not np.array_equal(a, oracle.run(L, q, POTTS, T, 2, 0, 7, s0))
    # init is uniform over the q states
    big = oracle.init_spins(256, 6, 5)
    cnt = np.bincount(big.reshape(-1), minlength=6)
    assert abs(cnt - 256 * 256 / 6).max() < 5 * math.sqrt(256 * 256 / 6)
