"""Pins of the oracle's derived doubles (eq.(2), (3), (5), (6); R11, R15) against things other
than themselves: closed forms on structured lattices, an independent route from the spins (complex unit vectors,
simplex vectors of the Potts order parameter) and exact enumeration of the Boltzmann distribution (CPU only)."""
from __future__ import annotations

import math

import numpy as np
import pytest

POTTS, CLOCK = 0, 1


def _hists(oracle, L, q, s, r=None):
    bh, sh = oracle.observables(L, q, s)
    return (bh, sh) if r is None else (bh, sh, oracle.correlation(L, q, s, r))


@pytest.mark.parametrize("L,q", [(8, 2), (12, 3), (12, 6), (16, 4)])
def test_uniform_lattice_closed_forms(oracle, L, q):
    N = L * L
    s = np.full((L, L), q - 1, dtype=np.uint8)
    bh, sh = _hists(oracle, L, q, s)
    assert oracle.potts_energy(L, bh) == 0.0                      # eq.(1): every bond satisfied
    assert oracle.potts_m2(q, sh) == float(N * N)                 # eq.(3): fully ordered
    assert oracle.clock_energy(q, bh) == -2.0 * N                 # eq.(4): 2N bonds of cos 0
    assert abs(oracle.clock_m(q, sh) - N) < 1e-9 * N
    for r in (1, L // 4, L // 2):
        assert oracle.g(q, oracle.correlation(L, q, s, r)) == 1.0  # eq.(5)
    rows = np.stack([sh, sh, sh])
    assert oracle.moment_ratio(q, rows) == 1.0                    # eq.(2): no fluctuation
    ch = np.stack([oracle.correlation(L, q, s, L // 2)] * 2)
    cq = np.stack([oracle.correlation(L, q, s, L // 4)] * 2)
    assert oracle.ratio_R(q, ch, cq) == 1.0                       # eq.(6)


def test_checkerboard_q2_closed_forms(oracle):
    L, q = 8, 2
    N = L * L
    y, x = np.mgrid[0:L, 0:L]
    s = ((x + y) % 2).astype(np.uint8)
    bh, sh = _hists(oracle, L, q, s)
    assert oracle.potts_energy(L, bh) == 2.0 * N                  # every bond broken
    assert oracle.potts_m2(q, sh) == 0.0                          # half / half
    assert abs(oracle.clock_energy(q, bh) - 2.0 * N) < 1e-9       # cos(pi) = -1 on every bond
    assert oracle.clock_m(q, sh) < 1e-9
    for r in range(1, L):
        assert abs(oracle.g(q, oracle.correlation(L, q, s, r)) - (-1.0) ** r) < 1e-12


@pytest.mark.parametrize("q", [2, 3, 4, 6, 16])
def test_m2_equals_the_simplex_vector_definition(oracle, q):
    """The Potts order parameter is the sum of N unit vectors e_a of a regular simplex, e_a . e_b = (q delta_ab - 1)/(q - 1);
    its squared length is eq.(3).  Built here from explicit vectors, not from eq.(3)."""
    rng = np.random.default_rng(q)
    # simplex vectors: centred standard basis of R^q, rescaled to unit length
    e = np.eye(q) - 1.0 / q
    e /= np.linalg.norm(e[0])
    assert abs(e[0] @ e[1] - (-1.0 / (q - 1))) < 1e-12
    for _ in range(5):
        n = rng.integers(0, 5000, size=q)
        m = (n[:, None] * e).sum(axis=0)
        assert abs(oracle.potts_m2(q, n) - float(m @ m)) <= 1e-9 * max(1.0, float(m @ m))
    assert oracle.potts_m2(q, np.full(q, 7)) == 0.0               # equal populations
    big = np.zeros(q, dtype=np.int64)
    big[0] = 1 << 28                                              # N = 2^28 (L = 16384): the integer numerator must not overflow
    assert oracle.potts_m2(q, big) == float(1 << 56)
    if q == 2:
        assert oracle.potts_m2(2, [300, 100]) == 200.0 ** 2       # Ising: M = n0 - n1


@pytest.mark.parametrize("L,q,r", [(8, 6, 2), (12, 4, 3), (9, 5, 4), (16, 6, 8)])
def test_clock_quantities_from_the_spins_directly(oracle, L, q, r):
    """Energy, |M| and G(r) recomputed from the configuration as complex unit vectors z = exp(2 pi i s / q)."""
    rng = np.random.default_rng(100 * L + q)
    s = rng.integers(0, q, size=(L, L), dtype=np.uint8)
    z = np.exp(2j * np.pi * s.astype(np.float64) / q)
    bh, sh, ch = _hists(oracle, L, q, s, r)
    e = -(np.real(z * np.conj(np.roll(z, -1, axis=1))).sum() + np.real(z * np.conj(np.roll(z, -1, axis=0))).sum())
    assert abs(oracle.clock_energy(q, bh) - e) < 1e-9 * L * L
    assert abs(oracle.clock_m(q, sh) - abs(z.sum())) < 1e-9 * L * L
    gr = (np.real(z * np.conj(np.roll(z, -r, axis=1))).sum() + np.real(z * np.conj(np.roll(z, -r, axis=0))).sum()) / (2.0 * L * L)
    assert abs(oracle.g(q, ch) - gr) < 1e-12
    assert oracle.potts_energy(L, bh) == float(2 * L * L - np.count_nonzero(s == np.roll(s, -1, axis=1)) - np.count_nonzero(s == np.roll(s, -1, axis=0)))


def test_moment_ratio_small_series(oracle):
    # q = 2: M^2 = (n0 - n1)^2 -> 1 and 16: <M^4> = (1 + 256) / 2, <M^2>^2 = (17 / 2)^2
    assert abs(oracle.moment_ratio(2, [[1, 0], [4, 0]]) - (257.0 / 2.0) / (8.5 * 8.5)) < 1e-15
    # a transposed (row / column) read of the series would give a different number
    assert abs(oracle.moment_ratio(2, [[4, 0], [1, 0], [0, 0]]) - (257.0 / 3.0) / ((17.0 / 3.0) ** 2)) < 1e-15


def test_ratio_R_small_series(oracle):
    # q = 2: G = (c0 - c1) / (c0 + c1).  rows: G_half = 0.5, 0.0; G_quarter = 1.0, 0.5 -> R = 0.25 / 0.75
    ch = [[3, 1], [2, 2]]
    cq = [[4, 0], [3, 1]]
    assert abs(oracle.ratio_R(2, ch, cq) - (0.25 / 0.75)) < 1e-15


def test_U_and_R_match_exact_enumeration_4x4(oracle):
    """q = 2 Potts on the 4x4 torus at Tc: U of eq.(2) and, for the q = 2 clock model at T = 1.5, R of eq.(6) with
    L/2 = 2 and L/4 = 1, by the exact sum over the 2^16 states, against long oracle runs."""
    L, q, n = 4, 2, 16
    states = ((np.arange(1 << n)[:, None] >> np.arange(n)[None, :]) & 1).astype(np.int64).reshape(-1, L, L)
    sig = 1 - 2 * states
    nn = (sig * np.roll(sig, -1, axis=2)).sum(axis=(1, 2)) + (sig * np.roll(sig, -1, axis=1)).sum(axis=(1, 2))
    # Potts eq.(1): H = -sum (delta - 1) = (2N - n_eq), n_eq = (2N + nn) / 2
    T = 1.0 / math.log(1.0 + math.sqrt(2.0))
    w = np.exp(((2 * n + nn) / 2.0 - 2 * n) / T)
    m2 = sig.sum(axis=(1, 2)).astype(np.float64) ** 2
    U_exact = float((w * m2 * m2).sum() / w.sum()) / float((w * m2).sum() / w.sum()) ** 2
    seed, sweeps = 0xABCDEF, 60000
    s = oracle.init_spins(L, q, seed)
    s = oracle.run(L, q, POTTS, T, seed, 0, 200, s)
    s, _, sr = oracle.run(L, q, POTTS, T, seed, 200, sweeps, s, record=True)
    U = oracle.moment_ratio(q, sr)
    blocks = [oracle.moment_ratio(q, b) for b in np.array_split(sr, 30)]
    err = np.std(blocks, ddof=1) / math.sqrt(len(blocks))
    assert abs(U - U_exact) < 5.0 * err + 2e-3, (U, U_exact, err)

    # clock q = 2: H = -sum cos(pi (s_i - s_j)) = -nn
    Tc = 1.5
    wc = np.exp((nn - nn.max()) / Tc)

    def g_of(r):
        return ((sig * np.roll(sig, -r, axis=2)).sum(axis=(1, 2)) + (sig * np.roll(sig, -r, axis=1)).sum(axis=(1, 2))) / (2.0 * n)

    R_exact = float((wc * g_of(2)).sum() / (wc * g_of(1)).sum())
    seed, sweeps = 0xC0FFEE, 40000
    s = oracle.init_spins(L, q, seed)
    s = oracle.run(L, q, CLOCK, Tc, seed, 0, 200, s)
    ch, cq = [], []
    for t in range(200, 200 + sweeps):
        ch.append(oracle.correlation(L, q, s, 2))
        cq.append(oracle.correlation(L, q, s, 1))
        s = oracle.run(L, q, CLOCK, Tc, seed, t, 1, s)
    ch, cq = np.array(ch), np.array(cq)
    R = oracle.ratio_R(q, ch, cq)
    blocks = [oracle.ratio_R(q, a, b) for a, b in zip(np.array_split(ch, 30), np.array_split(cq, 30))]
    err = np.std(blocks, ddof=1) / math.sqrt(len(blocks))
    assert abs(R - R_exact) < 5.0 * err + 2e-3, (R, R_exact, err)
