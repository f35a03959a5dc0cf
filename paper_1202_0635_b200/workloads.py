"""Seeded, synthetic workload descriptions shared by the tests, bench.py and smoke().

This module holds NO arithmetic of the method (no Philox, no thresholds, no labeling): only the
parameters of the paper's workloads (PAPER.md:75 -- q=2,3 Potts at Tc = 1/ln(1+sqrt q);
PAPER.md:142 -- q=6 clock at T = 0.9; BASELINE.json configs 1-5) and a few plain numpy
generators of spin configurations used to hand the same bytes to the oracle and to the CUDA path.
"""
from __future__ import annotations

import math
from dataclasses import dataclass

import numpy as np

POTTS = 0
CLOCK = 1


def potts_tc(q: int) -> float:
    """Tc/J of the q-state Potts model of PAPER.md eq.(1), as printed in PAPER.md:75."""
    return 1.0 / math.log(1.0 + math.sqrt(float(q)))


@dataclass(frozen=True)
class Workload:
    name: str
    L: int
    q: int
    model: int
    T: float
    seed: int
    sweeps: int          # run length the config names (not what a test or the bench executes)
    equil: int = 0       # sweeps before measurements start


# BASELINE.json "configs" 1..5 (config 4 and 5 expand to several rows).
CONFIGS = {
    "c1_potts2_L64": Workload("c1_potts2_L64", 64, 2, POTTS, potts_tc(2), 0x5EED0001, 1000),
    "c2_potts2_L4096": Workload("c2_potts2_L4096", 4096, 2, POTTS, potts_tc(2), 0x5EED0002, 10000, 1000),
    "c3_clock6_L4096": Workload("c3_clock6_L4096", 4096, 6, CLOCK, 0.9, 0x5EED0003, 10000),
    "c4_potts3_L8192": Workload("c4_potts3_L8192", 8192, 3, POTTS, potts_tc(3), 0x5EED0004, 5000),
    "c4_potts4_L8192": Workload("c4_potts4_L8192", 8192, 4, POTTS, potts_tc(4), 0x5EED1004, 5000),
    "c5_potts2_L16384_0.8Tc": Workload("c5_potts2_L16384_0.8Tc", 16384, 2, POTTS, 0.8 * potts_tc(2), 0x5EED0005, 1000),
    "c5_potts2_L16384_Tc": Workload("c5_potts2_L16384_Tc", 16384, 2, POTTS, 1.0 * potts_tc(2), 0x5EED1005, 1000),
    "c5_potts2_L16384_1.2Tc": Workload("c5_potts2_L16384_1.2Tc", 16384, 2, POTTS, 1.2 * potts_tc(2), 0x5EED2005, 1000),
}

# The workload BASELINE.json's metric is quoted on ("ns per spin flip (full SW sweep) at L=4096, T_c").
HEADLINE = "c2_potts2_L4096"


def random_spins(L: int, q: int, seed: int) -> np.ndarray:
    """Uniform random states from numpy's own generator (for sw_set_spins hand-offs)."""
    rng = np.random.default_rng(seed)
    return rng.integers(0, q, size=(L, L), dtype=np.uint8)


def uniform_spins(L: int, state: int) -> np.ndarray:
    return np.full((L, L), state, dtype=np.uint8)


def stripes(L: int, q: int, width: int, vertical: bool) -> np.ndarray:
    idx = np.arange(L) // max(1, width)
    row = (idx % q).astype(np.uint8)
    a = np.broadcast_to(row[None, :] if vertical else row[:, None], (L, L))
    return np.ascontiguousarray(a)


def checkerboard(L: int, q: int) -> np.ndarray:
    y, x = np.mgrid[0:L, 0:L]
    return ((x + y) % q).astype(np.uint8)


def domains(L: int, q: int, seed: int, block: int) -> np.ndarray:
    """Random states constant on block x block squares: large clusters with ragged seams."""
    rng = np.random.default_rng(seed)
    nb = (L + block - 1) // block
    coarse = rng.integers(0, q, size=(nb, nb), dtype=np.uint8)
    return np.ascontiguousarray(np.kron(coarse, np.ones((block, block), dtype=np.uint8))[:L, :L])
