"""One lattice sharded over ranks by row stripes (NEXT-3, scheme of SURVEY.md 8(e)): the exchange steps.

The arithmetic is in libsw.so (``sw_stripe_*`` kernels, ``sw_seam_solve`` host code); this module only moves the two small
messages of a sweep between ranks with ``torch.distributed`` (NCCL between GPUs, gloo on CPUs) or, for one process that
holds all stripes, through plain numpy -- and marshals the seam solve.  No method arithmetic here.

A sweep, per rank:  first rows all-gathered (L bytes each; rank r takes the row of rank r + 1 as its halo)  ->  label  ->
(first-row roots, last-row roots, seam bonds) all-gathered (9 L bytes each)  ->  seam solve, identical on every rank  ->
finish.
"""
from __future__ import annotations

import ctypes

import numpy as np

from . import binding as _b


def solve_seams(first: np.ndarray, last: np.ndarray, seam: np.ndarray):
    """sw_seam_solve on gathered [G][L] arrays -> (from, to): local roots and their canonical roots.  Host only."""
    first = np.ascontiguousarray(first, dtype=np.int32)
    last = np.ascontiguousarray(last, dtype=np.int32)
    seam = np.ascontiguousarray(seam, dtype=np.uint8)
    G, L = first.shape
    assert last.shape == (G, L) and seam.shape == (G, L)
    frm = np.zeros(2 * G * L, dtype=np.int32)
    to = np.zeros(2 * G * L, dtype=np.int32)
    n = ctypes.c_int(0)
    rc = _b.load().sw_seam_solve(G, L, first.ctypes.data, last.ctypes.data, seam.ctypes.data, frm.ctypes.data, to.ctypes.data, ctypes.byref(n))
    if rc != _b.SW_OK:
        raise _b.SwError(rc, "sw_seam_solve failed")
    return frm[: n.value].copy(), to[: n.value].copy()


class Stripe:
    """Rows [rank L / nranks, (rank + 1) L / nranks) of one L x L lattice on the current CUDA device."""

    def __init__(self, L: int, q: int, model: int, T: float, seed: int, rank: int, nranks: int):
        self._lib = _b.load()
        self.L, self.q, self.rank, self.nranks = L, q, rank, nranks
        self.rows = L // nranks
        h = self._lib.sw_stripe_create(L, q, model, float(T), seed, rank, nranks)
        if not h:
            raise _b.SwError(_b.SW_ERR_ARG, f"sw_stripe_create(L={L}, q={q}, rank={rank}/{nranks}) failed (needs a CUDA device, L % nranks == 0, L % 4 == 0)")
        self._h = h

    def close(self):
        if self._h:
            self._lib.sw_stripe_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def first_row(self) -> np.ndarray:
        out = np.empty(self.L, dtype=np.uint8)
        _b._check(self._lib.sw_stripe_first_row(self._h, out.ctypes.data))
        return out

    def label(self, halo_row: np.ndarray):
        halo_row = np.ascontiguousarray(halo_row, dtype=np.uint8)
        assert halo_row.size == self.L
        _b._check(self._lib.sw_stripe_label(self._h, halo_row.ctypes.data))

    def export_seam(self):
        first = np.empty(self.L, dtype=np.int32)
        last = np.empty(self.L, dtype=np.int32)
        seam = np.empty(self.L, dtype=np.uint8)
        _b._check(self._lib.sw_stripe_export_seam(self._h, first.ctypes.data, last.ctypes.data, seam.ctypes.data))
        return first, last, seam

    def finish(self, frm: np.ndarray, to: np.ndarray):
        frm = np.ascontiguousarray(frm, dtype=np.int32)
        to = np.ascontiguousarray(to, dtype=np.int32)
        _b._check(self._lib.sw_stripe_finish(self._h, int(frm.size), frm.ctypes.data, to.ctypes.data))

    def get_spins(self) -> np.ndarray:
        out = np.empty((self.rows, self.L), dtype=np.uint8)
        _b._check(self._lib.sw_stripe_get_spins(self._h, out.ctypes.data))
        return out

    def get_labels(self) -> np.ndarray:
        out = np.empty((self.rows, self.L), dtype=np.int32)
        _b._check(self._lib.sw_stripe_get_labels(self._h, out.ctypes.data))
        return out

    def set_spins(self, spins: np.ndarray, sweep_index: int):
        spins = np.ascontiguousarray(spins, dtype=np.uint8)
        assert spins.size == self.rows * self.L
        _b._check(self._lib.sw_stripe_set_spins(self._h, spins.ctypes.data, sweep_index))

    @property
    def sweep_index(self) -> int:
        return int(self._lib.sw_stripe_sweep_index(self._h))


def sweep_local(stripes):
    """One sweep of ALL stripes held by this process (one GPU standing in for G ranks, one stripe after the other: no
    kernel waits on another).  The same message flow as sweep_distributed, through numpy."""
    G = len(stripes)
    rows = [s.first_row() for s in stripes]
    for g, s in enumerate(stripes):
        s.label(rows[(g + 1) % G])
    exp = [s.export_seam() for s in stripes]
    frm, to = solve_seams(np.stack([e[0] for e in exp]), np.stack([e[1] for e in exp]), np.stack([e[2] for e in exp]))
    for s in stripes:
        s.finish(frm, to)


def gather_rows(row: np.ndarray, dist, device: str = "cpu") -> np.ndarray:
    """all_gather of one fixed-size numpy row per rank -> [world][len] (torch.distributed plumbing)."""
    import torch
    t = torch.from_numpy(np.ascontiguousarray(row)).to(device)
    out = [torch.empty_like(t) for _ in range(dist.get_world_size())]
    dist.all_gather(out, t)
    return np.stack([o.cpu().numpy() for o in out])


def sweep_distributed(stripe, dist, device: str = "cuda"):
    """One sweep of this rank's stripe inside an initialised torch.distributed group (NCCL: device='cuda')."""
    rank, G = dist.get_rank(), dist.get_world_size()
    rows = gather_rows(stripe.first_row(), dist, device)
    stripe.label(rows[(rank + 1) % G])
    first, last, seam = stripe.export_seam()
    frm, to = solve_seams(gather_rows(first, dist, device), gather_rows(last, dist, device), gather_rows(seam, dist, device))
    stripe.finish(frm, to)
