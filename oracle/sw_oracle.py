"""ctypes loader for the C oracle (``oracle/sw_oracle.c``).

ORACLE = test infrastructure, not the product.  Only ``tests/``, ``__graft_entry__.smoke()`` and
``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs may import this module.  It never
imports the CUDA package and shares nothing with it.

``build()`` compiles the C file with ``gcc -O2`` into ``oracle/libsw_oracle.so`` (git-ignored).
Every wrapper below only marshals numpy arrays; all arithmetic is in the C file, which cites
PAPER.md for each step.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "sw_oracle.c"
_LIB = _HERE / "libsw_oracle.so"

POTTS = 0
CLOCK = 1

_u8p = ctypes.POINTER(ctypes.c_uint8)
_i32p = ctypes.POINTER(ctypes.c_int32)
_u32p = ctypes.POINTER(ctypes.c_uint32)
_i64p = ctypes.POINTER(ctypes.c_int64)


def build(force: bool = False) -> Path:
    """Compile the oracle if the shared object is missing or older than the source."""
    if force or not _LIB.exists() or _LIB.stat().st_mtime < _SRC.stat().st_mtime:
        tmp = _LIB.with_suffix(f".so.tmp{os.getpid()}")
        subprocess.run(
            ["gcc", "-O2", "-std=c99", "-fPIC", "-shared", "-o", str(tmp), str(_SRC), "-lm"],
            check=True,
        )
        os.replace(tmp, _LIB)
    return _LIB


_lib = None


def lib() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        build()
        L = ctypes.CDLL(str(_LIB))
        L.oracle_philox4x32_10.argtypes = [_u32p, _u32p, _u32p]
        L.oracle_philox4x32_10.restype = None
        L.oracle_axis.argtypes = [ctypes.c_int, ctypes.c_uint64, ctypes.c_uint32]
        L.oracle_axis.restype = ctypes.c_uint32
        L.oracle_potts_threshold.argtypes = [ctypes.c_double]
        L.oracle_potts_threshold.restype = ctypes.c_uint32
        L.oracle_clock_table.argtypes = [ctypes.c_int, ctypes.c_double, _u32p]
        L.oracle_clock_table.restype = None
        L.oracle_init_spins.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_uint64, _u8p]
        L.oracle_init_spins.restype = None
        L.oracle_bonds.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_double,
                                   ctypes.c_uint64, ctypes.c_uint32, _u8p, _u8p]
        L.oracle_bonds.restype = ctypes.c_int
        L.oracle_label.argtypes = [ctypes.c_int, _u8p, _i32p]
        L.oracle_label.restype = None
        L.oracle_flip.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_uint64,
                                  ctypes.c_uint32, _i32p, _u8p]
        L.oracle_flip.restype = None
        L.oracle_sweep.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_double,
                                   ctypes.c_uint64, ctypes.c_uint32, _u8p, _i32p, _u8p]
        L.oracle_sweep.restype = ctypes.c_int
        L.oracle_observables.argtypes = [ctypes.c_int, ctypes.c_int, _u8p, _i64p, _i64p]
        L.oracle_observables.restype = None
        L.oracle_correlation.argtypes = [ctypes.c_int, ctypes.c_int, _u8p, ctypes.c_int, _i64p]
        L.oracle_correlation.restype = None
        L.oracle_run.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_double,
                                 ctypes.c_uint64, ctypes.c_uint32, ctypes.c_int, _u8p, _i64p, _i64p]
        L.oracle_run.restype = ctypes.c_int
        for name, args in (("oracle_potts_energy", [ctypes.c_int, _i64p]), ("oracle_potts_m2", [ctypes.c_int, _i64p]),
                           ("oracle_clock_energy", [ctypes.c_int, _i64p]), ("oracle_clock_m", [ctypes.c_int, _i64p]),
                           ("oracle_g", [ctypes.c_int, _i64p]), ("oracle_moment_ratio", [ctypes.c_int, ctypes.c_int, _i64p]),
                           ("oracle_ratio_R", [ctypes.c_int, ctypes.c_int, _i64p, _i64p])):
            fn = getattr(L, name)
            fn.argtypes = args
            fn.restype = ctypes.c_double
        _lib = L
    return _lib


def _p(a: np.ndarray, typ):
    return a.ctypes.data_as(typ)


def philox4x32_10(ctr, key) -> np.ndarray:
    c = np.ascontiguousarray(ctr, dtype=np.uint32)
    k = np.ascontiguousarray(key, dtype=np.uint32)
    assert c.shape == (4,) and k.shape == (2,)
    out = np.zeros(4, dtype=np.uint32)
    lib().oracle_philox4x32_10(_p(c, _u32p), _p(k, _u32p), _p(out, _u32p))
    return out


def axis(q: int, seed: int, t: int) -> int:
    return int(lib().oracle_axis(q, seed, t))


def potts_threshold(T: float) -> int:
    return int(lib().oracle_potts_threshold(float(T)))


def clock_table(q: int, T: float) -> np.ndarray:
    tab = np.zeros((2 * q, 2 * q), dtype=np.uint32)
    lib().oracle_clock_table(q, float(T), _p(tab, _u32p))
    return tab


def thresholds(q: int, model: int, T: float) -> np.ndarray:
    """The threshold export in the boundary's format: 1 word (Potts) or (2q)^2 words (clock)."""
    if model == POTTS:
        return np.array([potts_threshold(T)], dtype=np.uint32)
    return clock_table(q, T).reshape(-1)


def init_spins(L: int, q: int, seed: int) -> np.ndarray:
    s = np.zeros((L, L), dtype=np.uint8)
    lib().oracle_init_spins(L, q, seed, _p(s, _u8p))
    return s


def bonds(L, q, model, T, seed, t, spins) -> np.ndarray:
    s = np.ascontiguousarray(spins, dtype=np.uint8).reshape(L, L)
    b = np.zeros((L, L), dtype=np.uint8)
    rc = lib().oracle_bonds(L, q, model, float(T), seed, t, _p(s, _u8p), _p(b, _u8p))
    assert rc == 0
    return b


def label(L, bonds_arr) -> np.ndarray:
    b = np.ascontiguousarray(bonds_arr, dtype=np.uint8).reshape(L, L)
    lab = np.zeros((L, L), dtype=np.int32)
    lib().oracle_label(L, _p(b, _u8p), _p(lab, _i32p))
    return lab


def flip(L, q, model, seed, t, labels, spins) -> np.ndarray:
    lab = np.ascontiguousarray(labels, dtype=np.int32).reshape(L, L)
    s = np.array(spins, dtype=np.uint8, copy=True).reshape(L, L)
    lib().oracle_flip(L, q, model, seed, t, _p(lab, _i32p), _p(s, _u8p))
    return s


def sweep(L, q, model, T, seed, t, spins, want_labels=False, want_bonds=False):
    """One sweep t on a copy of ``spins``; returns new spins (and labels / bonds if asked)."""
    s = np.array(spins, dtype=np.uint8, copy=True).reshape(L, L)
    lab = np.zeros((L, L), dtype=np.int32) if want_labels else None
    bnd = np.zeros((L, L), dtype=np.uint8) if want_bonds else None
    rc = lib().oracle_sweep(L, q, model, float(T), seed, t, _p(s, _u8p),
                            _p(lab, _i32p) if want_labels else None,
                            _p(bnd, _u8p) if want_bonds else None)
    assert rc == 0
    out = [s]
    if want_labels:
        out.append(lab)
    if want_bonds:
        out.append(bnd)
    return out[0] if len(out) == 1 else tuple(out)


def observables(L, q, spins):
    s = np.ascontiguousarray(spins, dtype=np.uint8).reshape(L, L)
    bh = np.zeros(q, dtype=np.int64)
    sh = np.zeros(q, dtype=np.int64)
    lib().oracle_observables(L, q, _p(s, _u8p), _p(bh, _i64p), _p(sh, _i64p))
    return bh, sh


def correlation(L, q, spins, r):
    """corr_hist[d] = #{pairs at distance r along +x and +y with (S_i - S_j) mod q == d} (eq.(5); R15)."""
    s = np.ascontiguousarray(spins, dtype=np.uint8).reshape(L, L)
    ch = np.zeros(q, dtype=np.int64)
    lib().oracle_correlation(L, q, _p(s, _u8p), int(r), _p(ch, _i64p))
    return ch


def _i64(a, shape=None) -> np.ndarray:
    a = np.ascontiguousarray(a, dtype=np.int64)
    if shape is not None:
        a = a.reshape(shape)
    return a


def potts_energy(L, bond_hist) -> float:
    return float(lib().oracle_potts_energy(L, _p(_i64(bond_hist), _i64p)))


def potts_m2(q, state_hist) -> float:
    return float(lib().oracle_potts_m2(q, _p(_i64(state_hist), _i64p)))


def clock_energy(q, bond_hist) -> float:
    return float(lib().oracle_clock_energy(q, _p(_i64(bond_hist), _i64p)))


def clock_m(q, state_hist) -> float:
    return float(lib().oracle_clock_m(q, _p(_i64(state_hist), _i64p)))


def g(q, corr_hist) -> float:
    return float(lib().oracle_g(q, _p(_i64(corr_hist), _i64p)))


def moment_ratio(q, state_hist_rows) -> float:
    rows = _i64(state_hist_rows, (-1, q))
    return float(lib().oracle_moment_ratio(rows.shape[0], q, _p(rows, _i64p)))


def ratio_R(q, corr_half_rows, corr_quarter_rows) -> float:
    a, b = _i64(corr_half_rows, (-1, q)), _i64(corr_quarter_rows, (-1, q))
    assert a.shape == b.shape
    return float(lib().oracle_ratio_R(a.shape[0], q, _p(a, _i64p), _p(b, _i64p)))


def run(L, q, model, T, seed, t0, n, spins, record=False):
    """n sweeps t0..t0+n-1 on a copy of ``spins``.  With record=True also returns the per-sweep
    (bond_hist, state_hist) rows, row k = configuration BEFORE sweep t0+k."""
    s = np.array(spins, dtype=np.uint8, copy=True).reshape(L, L)
    if record:
        br = np.zeros((n, q), dtype=np.int64)
        sr = np.zeros((n, q), dtype=np.int64)
        rc = lib().oracle_run(L, q, model, float(T), seed, t0, n, _p(s, _u8p), _p(br, _i64p), _p(sr, _i64p))
        assert rc == 0
        return s, br, sr
    rc = lib().oracle_run(L, q, model, float(T), seed, t0, n, _p(s, _u8p), None, None)
    assert rc == 0
    return s
