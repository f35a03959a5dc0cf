"""Pins of oracle_correlation (eq.(5), (6); R15) against things other than itself (CPU only)."""
from __future__ import annotations

import math

import numpy as np
import pytest

CLOCK = 1


@pytest.mark.parametrize("L,q", [(4, 2), (6, 3), (8, 6), (9, 5)])
def test_distance_one_is_the_bond_histogram(oracle, L, q):
    rng = np.random.default_rng(7 * L + q)
    s = rng.integers(0, q, size=(L, L), dtype=np.uint8)
    bh, _ = oracle.observables(L, q, s)          # a different function of the oracle (pinned on its own)
    assert np.array_equal(oracle.correlation(L, q, s, 1), bh)


@pytest.mark.parametrize("L,q,r", [(8, 6, 2), (8, 6, 4), (12, 4, 3), (12, 4, 6), (5, 3, 2)])
def test_roll_restatement_symmetry_and_sums(oracle, L, q, r):
    rng = np.random.default_rng(L + 100 * r + q)
    s = rng.integers(0, q, size=(L, L), dtype=np.uint8)
    ch = oracle.correlation(L, q, s, r)
    si = s.astype(np.int64)
    d = np.concatenate([((si - np.roll(si, -r, axis=1)) % q).ravel(), ((si - np.roll(si, -r, axis=0)) % q).ravel()])
    assert np.array_equal(ch, np.bincount(d, minlength=q))
    assert ch.sum() == 2 * L * L
    back = oracle.correlation(L, q, s, L - r)    # the same pairs seen from the other end: d -> -d
    assert np.array_equal(back, ch[(-np.arange(q)) % q])
    zero = oracle.correlation(L, q, s, 0)
    assert zero[0] == 2 * L * L and zero[1:].sum() == 0


def test_stripes_closed_form(oracle):
    L, q, w = 24, 6, 2
    x = np.arange(L)
    s = np.broadcast_to(((x // w) % q).astype(np.uint8), (L, L)).copy()   # vertical stripes of width 2, states cycling
    for r in (2, 4, 6, 12):
        ch = oracle.correlation(L, q, s, r)
        expect = np.zeros(q, dtype=np.int64)
        expect[0] += L * L                       # along y every pair is equal
        expect[(-(r // w)) % q] += L * L         # along x the state advances by r / w (L / w = 12 is a multiple of q)
        assert np.array_equal(ch, expect), r


def test_long_run_matches_exact_enumeration_4x4(oracle):
    """<cos(2 pi (S_i - S_{i+2}) / q)> of the q=2 clock model on the 4x4 torus, T = 1.5: exact sum over the 2^16 states
    of the Boltzmann weight of PAPER.md eq.(4) against the average over an oracle run (pins the r indexing and, once
    more, the clock sweep)."""
    L, q, T, r = 4, 2, 1.5, 2
    n = L * L
    states = ((np.arange(1 << n)[:, None] >> np.arange(n)[None, :]) & 1).astype(np.int64).reshape(-1, L, L)
    sig = 1 - 2 * states                                             # cos(pi s) = +-1
    e = -(sig * np.roll(sig, -1, axis=2)).sum(axis=(1, 2)) - (sig * np.roll(sig, -1, axis=1)).sum(axis=(1, 2))
    w = np.exp(-(e - e.min()) / T)
    g = ((sig * np.roll(sig, -r, axis=2)).sum(axis=(1, 2)) + (sig * np.roll(sig, -r, axis=1)).sum(axis=(1, 2))) / (2.0 * n)
    exact = float((w * g).sum() / w.sum())
    seed, sweeps = 0xC0FFEE, 40000
    s = oracle.init_spins(L, q, seed)
    s = oracle.run(L, q, CLOCK, T, seed, 0, 200, s)
    acc = []
    for t in range(200, 200 + sweeps):
        ch = oracle.correlation(L, q, s, r)
        acc.append((ch[0] - ch[1]) / (2.0 * n))
        s = oracle.run(L, q, CLOCK, T, seed, t, 1, s)
    acc = np.array(acc)
    blocks = acc[: len(acc) // 50 * 50].reshape(50, -1).mean(axis=1)
    err = blocks.std(ddof=1) / math.sqrt(len(blocks))
    assert abs(acc.mean() - exact) < 5.0 * err + 1e-4, (acc.mean(), exact, err)
