"""Thin ctypes binding of ``include/sw.h`` (libsw.so).  Argument marshalling only.

Every step of the sweep runs in the CUDA kernels of ``csrc/``; this module never computes anything
of the method and has no CPU fallback: loading fails loudly if ``libsw.so`` has not been built
(``python -m paper_1202_0635_b200.build`` or ``__graft_entry__.build()``), and every call fails
with ``SwError`` if no CUDA device is usable.

PyTorch is used for plumbing only: ``Lattice`` gets its device workspace from ``torch.empty`` and
runs on the current torch CUDA stream (``sw_create_in``), so ``torch.cuda.Event`` timing on that
stream sees the kernels.
"""
from __future__ import annotations

import ctypes
import os
from pathlib import Path

import numpy as np

_PKG = Path(__file__).resolve().parent
# SW_LIB: load another build of the same library (tests/test_gpu_parity.py builds one with tiny list capacities)
LIB_PATH = Path(os.environ["SW_LIB"]) if os.environ.get("SW_LIB") else _PKG / "libsw.so"

SW_POTTS, SW_CLOCK = 0, 1
SW_OK, SW_ERR_ARG, SW_ERR_CUDA, SW_ERR_NOMEM, SW_ERR_UNSUPPORTED = 0, -1, -2, -3, -4
SW_ALGO_AUTO, SW_ALGO_GENERIC, SW_ALGO_TILED, SW_ALGO_SMALL, SW_ALGO_HAWICK, SW_ALGO_KALENTEV = 0, 1, 2, 3, 4, 5

# name -> (restype, argtypes): every symbol include/sw.h declares
_vp, _i, _u64, _d, _sz = ctypes.c_void_p, ctypes.c_int, ctypes.c_uint64, ctypes.c_double, ctypes.c_size_t
SYMBOLS = {
    "sw_workspace_bytes": (_sz, [_i, _i, _i]),
    "sw_create": (_vp, [_i, _i, _i, _d, _u64]),
    "sw_create_in": (_vp, [_i, _i, _i, _d, _u64, _vp, _sz, _vp]),
    "sw_destroy": (None, [_vp]),
    "sw_sweep": (_i, [_vp, _i]),
    "sw_sweep_async": (_i, [_vp, _i]),
    "sw_sync": (_i, [_vp]),
    "sw_sweep_record": (_i, [_vp, _i, _vp, _vp]),
    "sw_observables": (_i, [_vp, _vp, _vp]),
    "sw_correlation": (_i, [_vp, _i, _vp]),
    "sw_sweep_record_corr": (_i, [_vp, _i, _i, _i, _vp, _vp, _vp, _vp]),
    "sw_get_spins": (_i, [_vp, _vp]),
    "sw_set_spins": (_i, [_vp, _vp, _u64]),
    "sw_sweep_index": (_u64, [_vp]),
    "sw_get_thresholds": (_i, [_vp, _vp, ctypes.POINTER(_i)]),
    "sw_get_labels": (_i, [_vp, _vp]),
    "sw_debug_bonds": (_i, [_vp, _vp]),
    "sw_set_algorithm": (_i, [_vp, _i]),
    "sw_get_algorithm": (_i, [_vp]),
    "sw_enable_stats": (_i, [_vp, _i]),
    "sw_stats": (_i, [_vp, _vp]),
    "sw_sweep_profile": (_i, [_vp, _i, _vp, ctypes.POINTER(_i)]),
    "sw_kernel_name": (ctypes.c_char_p, [_vp, _i]),
    "sw_launch_count": (_u64, [_vp]),
    "sw_derive_potts_energy": (_d, [_i, _vp]),
    "sw_derive_potts_m2": (_d, [_i, _vp]),
    "sw_derive_clock_energy": (_d, [_i, _vp]),
    "sw_derive_clock_m": (_d, [_i, _vp]),
    "sw_derive_g": (_d, [_i, _vp]),
    "sw_derive_moment_ratio": (_d, [_i, _i, _vp]),
    "sw_derive_ratio_R": (_d, [_i, _i, _vp, _vp]),
    "sw_create_batch": (_vp, [_i, _i, _i, _i, _vp, _vp]),
    "sw_batch_destroy": (None, [_vp]),
    "sw_batch_sweep": (_i, [_vp, _i]),
    "sw_batch_get_spins": (_i, [_vp, _vp]),
    "sw_batch_set_spins": (_i, [_vp, _vp, _u64]),
    "sw_batch_observables": (_i, [_vp, _vp, _vp]),
    "sw_batch_sweep_index": (_u64, [_vp]),
    "sw_stripe_create": (_vp, [_i, _i, _i, _d, _u64, _i, _i]),
    "sw_stripe_destroy": (None, [_vp]),
    "sw_stripe_first_row": (_i, [_vp, _vp]),
    "sw_stripe_label": (_i, [_vp, _vp]),
    "sw_stripe_export_seam": (_i, [_vp, _vp, _vp, _vp]),
    "sw_seam_solve": (_i, [_i, _i, _vp, _vp, _vp, _vp, _vp, ctypes.POINTER(_i)]),
    "sw_stripe_finish": (_i, [_vp, _i, _vp, _vp]),
    "sw_stripe_get_spins": (_i, [_vp, _vp]),
    "sw_stripe_get_labels": (_i, [_vp, _vp]),
    "sw_stripe_set_spins": (_i, [_vp, _vp, _u64]),
    "sw_stripe_sweep_index": (_u64, [_vp]),
    "sw_microbench": (_i, [_i, _i, _i, _vp]),
    "sw_microbench_name": (ctypes.c_char_p, [_i]),
    "sw_selftest": (_i, []),
    "sw_sweep_noalloc": (_i, [_i, _i, _i, _d, _u64, _u64, _vp, _vp, _vp]),
    "sw_last_error": (ctypes.c_char_p, []),
}


class SwError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"libsw error {code}: {msg}")
        self.code = code


_lib = None


def load() -> ctypes.CDLL:
    """Load libsw.so (no GPU needed to load; needed for any compute call)."""
    global _lib
    if _lib is None:
        if not LIB_PATH.exists():
            raise ImportError(
                f"{LIB_PATH} is missing: build the CUDA extension first "
                "(python -m paper_1202_0635_b200.build). There is no CPU fallback.")
        lib = ctypes.CDLL(str(LIB_PATH))
        for name, (res, args) in SYMBOLS.items():
            fn = getattr(lib, name)
            fn.restype = res
            fn.argtypes = args
        _lib = lib
    return _lib


def last_error() -> str:
    return load().sw_last_error().decode()


def _check(rc: int):
    if rc != SW_OK:
        raise SwError(rc, last_error())


def _host_ptr(a) -> int:
    """Pointer of a host buffer: numpy array or CPU torch tensor (pinned or not)."""
    if isinstance(a, np.ndarray):
        assert a.flags["C_CONTIGUOUS"]
        return a.ctypes.data
    return a.data_ptr()  # torch CPU tensor


class Lattice:
    """One SW context.  Methods mirror the C entry points one to one."""

    def __init__(self, L: int, q: int, model: int, T: float, seed: int, algo: int = SW_ALGO_AUTO,
                 torch_memory: bool = True):
        lib = load()
        self._lib = lib
        self.L, self.q, self.model, self.T, self.seed = L, q, model, float(T), seed
        self._ws = None
        self._h = None
        if torch_memory:
            import torch
            if not torch.cuda.is_available():
                raise SwError(SW_ERR_CUDA, "no CUDA device: the SW path has no CPU fallback")
            nbytes = lib.sw_workspace_bytes(L, q, model)
            if nbytes == 0:
                raise SwError(SW_ERR_ARG, f"invalid arguments L={L} q={q} model={model}")
            self._ws = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
            self.stream = torch.cuda.current_stream()
            h = lib.sw_create_in(L, q, model, self.T, seed, self._ws.data_ptr(), nbytes, self.stream.cuda_stream)
        else:
            h = lib.sw_create(L, q, model, self.T, seed)
        if not h:
            raise SwError(SW_ERR_ARG, last_error())
        self._h = h
        if algo != SW_ALGO_AUTO:
            self.set_algorithm(algo)

    # -- lifetime -------------------------------------------------------------------------------
    def close(self):
        if self._h:
            self._lib.sw_destroy(self._h)
            self._h = None
            self._ws = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    # -- the boundary ---------------------------------------------------------------------------
    def sweep(self, n: int = 1):
        _check(self._lib.sw_sweep(self._h, n))

    def sweep_async(self, n: int = 1):
        _check(self._lib.sw_sweep_async(self._h, n))

    def sync(self):
        _check(self._lib.sw_sync(self._h))

    def sweep_record(self, n: int):
        bh = np.zeros((n, self.q), dtype=np.int64)
        sh = np.zeros((n, self.q), dtype=np.int64)
        _check(self._lib.sw_sweep_record(self._h, n, bh.ctypes.data, sh.ctypes.data))
        return bh, sh

    def sweep_record_corr(self, n: int, r1: int, r2: int):
        out = [np.zeros((n, self.q), dtype=np.int64) for _ in range(4)]
        _check(self._lib.sw_sweep_record_corr(self._h, n, int(r1), int(r2), *[a.ctypes.data for a in out]))
        return tuple(out)

    def correlation(self, r: int):
        ch = np.zeros(self.q, dtype=np.int64)
        _check(self._lib.sw_correlation(self._h, int(r), ch.ctypes.data))
        return ch

    def observables(self):
        bh = np.zeros(self.q, dtype=np.int64)
        sh = np.zeros(self.q, dtype=np.int64)
        _check(self._lib.sw_observables(self._h, bh.ctypes.data, sh.ctypes.data))
        return bh, sh

    def get_spins(self, out=None):
        if out is None:
            out = np.empty((self.L, self.L), dtype=np.uint8)
        _check(self._lib.sw_get_spins(self._h, _host_ptr(out)))
        return out

    def set_spins(self, spins, sweep_index: int = 0):
        if isinstance(spins, np.ndarray):
            spins = np.ascontiguousarray(spins, dtype=np.uint8)
            assert spins.size == self.L * self.L
        _check(self._lib.sw_set_spins(self._h, _host_ptr(spins), sweep_index))

    @property
    def sweep_index(self) -> int:
        return int(self._lib.sw_sweep_index(self._h))

    def get_thresholds(self) -> np.ndarray:
        n = ctypes.c_int(0)
        _check(self._lib.sw_get_thresholds(self._h, None, ctypes.byref(n)))
        out = np.zeros(n.value, dtype=np.uint32)
        _check(self._lib.sw_get_thresholds(self._h, out.ctypes.data, ctypes.byref(n)))
        return out

    def get_labels(self) -> np.ndarray:
        out = np.empty((self.L, self.L), dtype=np.int32)
        _check(self._lib.sw_get_labels(self._h, out.ctypes.data))
        return out

    def debug_bonds(self) -> np.ndarray:
        out = np.empty((self.L, self.L), dtype=np.uint8)
        _check(self._lib.sw_debug_bonds(self._h, out.ctypes.data))
        return out

    def set_algorithm(self, algo: int):
        _check(self._lib.sw_set_algorithm(self._h, algo))

    @property
    def algorithm(self) -> int:
        return int(self._lib.sw_get_algorithm(self._h))

    def enable_stats(self, on: bool = True):
        _check(self._lib.sw_enable_stats(self._h, 1 if on else 0))

    def stats(self) -> np.ndarray:
        out = np.zeros(16, dtype=np.float64)
        _check(self._lib.sw_stats(self._h, out.ctypes.data))
        return out

    def sweep_profile(self, n: int) -> dict:
        """n sweeps with per-kernel CUDA-event timing: {kernel name: summed ms over the n sweeps}."""
        ms = np.zeros(8, dtype=np.float64)
        nk = ctypes.c_int(0)
        _check(self._lib.sw_sweep_profile(self._h, n, ms.ctypes.data, ctypes.byref(nk)))
        return {self._lib.sw_kernel_name(self._h, k).decode(): float(ms[k]) for k in range(nk.value)}

    @property
    def launch_count(self) -> int:
        return int(self._lib.sw_launch_count(self._h))


class Batch:
    """B independent lattices (own T and seed each) advanced together; mirrors sw_create_batch / sw_batch_*."""

    def __init__(self, L: int, q: int, model: int, T, seed):
        lib = load()
        self._lib = lib
        self._T = np.ascontiguousarray(T, dtype=np.float64)
        self._seed = np.ascontiguousarray(seed, dtype=np.uint64)
        assert self._T.shape == self._seed.shape and self._T.ndim == 1
        self.B, self.L, self.q, self.model = int(self._T.shape[0]), L, q, model
        h = lib.sw_create_batch(self.B, L, q, model, self._T.ctypes.data, self._seed.ctypes.data)
        if not h:
            raise SwError(SW_ERR_ARG, last_error())
        self._h = h

    def close(self):
        if self._h:
            self._lib.sw_batch_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def sweep(self, n: int = 1):
        _check(self._lib.sw_batch_sweep(self._h, n))

    def get_spins(self) -> np.ndarray:
        out = np.empty((self.B, self.L, self.L), dtype=np.uint8)
        _check(self._lib.sw_batch_get_spins(self._h, out.ctypes.data))
        return out

    def set_spins(self, spins, sweep_index: int = 0):
        spins = np.ascontiguousarray(spins, dtype=np.uint8)
        assert spins.size == self.B * self.L * self.L
        _check(self._lib.sw_batch_set_spins(self._h, spins.ctypes.data, sweep_index))

    def observables(self):
        bh = np.zeros((self.B, self.q), dtype=np.int64)
        sh = np.zeros((self.B, self.q), dtype=np.int64)
        _check(self._lib.sw_batch_observables(self._h, bh.ctypes.data, sh.ctypes.data))
        return bh, sh

    @property
    def sweep_index(self) -> int:
        return int(self._lib.sw_batch_sweep_index(self._h))


SW_NOALLOC_MAX_L = 1024


def sweep_noalloc(L: int, q: int, model: int, T: float, seed: int, sweep_index: int, d_spins_in, d_spins_out, stream=None):
    """sw_sweep_noalloc: one sweep from/to DEVICE buffers (torch CUDA uint8 tensors or raw device pointers), scratch in
    the library's static device array, no allocation.  Asynchronous on `stream` (a raw cudaStream_t, default: torch's
    current stream); synchronise before reading the output."""
    def dev_ptr(a):
        return int(a) if isinstance(a, int) else a.data_ptr()
    if stream is None:
        import torch
        stream = torch.cuda.current_stream().cuda_stream
    _check(load().sw_sweep_noalloc(L, q, model, float(T), seed, sweep_index, dev_ptr(d_spins_in), dev_ptr(d_spins_out), stream))


# Derived doubles (R11, R15): computed by libsw.so (sw_derive_*), marshalled here.
def _i64(a, q=None) -> np.ndarray:
    a = np.ascontiguousarray(a, dtype=np.int64)
    return a if q is None else a.reshape(-1, q)


def potts_energy(L: int, bond_hist) -> float:
    return float(load().sw_derive_potts_energy(L, _i64(bond_hist).ctypes.data))


def potts_m2(q: int, state_hist) -> float:
    return float(load().sw_derive_potts_m2(q, _i64(state_hist).ctypes.data))


def clock_energy(q: int, bond_hist) -> float:
    return float(load().sw_derive_clock_energy(q, _i64(bond_hist).ctypes.data))


def clock_m(q: int, state_hist) -> float:
    return float(load().sw_derive_clock_m(q, _i64(state_hist).ctypes.data))


def g(q: int, corr_hist) -> float:
    return float(load().sw_derive_g(q, _i64(corr_hist).ctypes.data))


def moment_ratio(q: int, state_hist_rows) -> float:
    rows = _i64(state_hist_rows, q)
    return float(load().sw_derive_moment_ratio(rows.shape[0], q, rows.ctypes.data))


def ratio_R(q: int, corr_half_rows, corr_quarter_rows) -> float:
    a, b = _i64(corr_half_rows, q), _i64(corr_quarter_rows, q)
    assert a.shape == b.shape
    return float(load().sw_derive_ratio_R(a.shape[0], q, a.ctypes.data, b.ctypes.data))
