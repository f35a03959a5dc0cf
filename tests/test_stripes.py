"""NEXT-3: one lattice sharded by row stripes.

CPU (-m "not gpu"): the host side -- sw_seam_solve through the C ABI (needs no device) and the torch.distributed message
flow over gloo with world_size 2 -- reproduces the oracle's GLOBAL labels from per-stripe label sets.  The per-stripe labels
of that test come from the oracle's bonds and a plain numpy flood fill (test infrastructure, not the product).
GPU (-m gpu): G stripes held by one process, one after the other on one GPU, against the oracle sweep by sweep.
"""
from __future__ import annotations

import math
import os
import socket

import numpy as np
import pytest

POTTS, CLOCK = 0, 1


def tc(q):
    return 1.0 / math.log(1.0 + math.sqrt(float(q)))


def _stripe_local_labels(bonds, row0, rows, L):
    """Labels inside one stripe (rows row0 .. row0 + rows - 1), +y bonds of its last row left out; label = smallest GLOBAL
    site index of the piece.  Plain flood fill."""
    lab = -np.ones((rows, L), dtype=np.int64)
    for y0 in range(rows):
        for x0 in range(L):
            if lab[y0, x0] >= 0:
                continue
            root = (row0 + y0) * L + x0              # scan order: the first unvisited site of a piece is its minimum
            stack = [(y0, x0)]
            lab[y0, x0] = root
            while stack:
                y, x = stack.pop()
                b = bonds[row0 + y, x]
                nb = []
                if b & 1:
                    nb.append((y, (x + 1) % L))
                if bonds[row0 + y, (x - 1) % L] & 1:
                    nb.append((y, (x - 1) % L))
                if (b & 2) and y + 1 < rows:
                    nb.append((y + 1, x))
                if y > 0 and (bonds[row0 + y - 1, x] & 2):
                    nb.append((y - 1, x))
                for (yy, xx) in nb:
                    if lab[yy, xx] < 0:
                        lab[yy, xx] = root
                        stack.append((yy, xx))
    return lab.astype(np.int32)


def _apply(lab, frm, to):
    out = lab.copy()
    for f, t in zip(frm, to):
        out[lab == f] = t
    return out


@pytest.mark.parametrize("L,G,q,T", [(16, 2, 2, tc(2)), (24, 4, 2, 0.8 * tc(2)), (32, 2, 3, tc(3)), (16, 8, 2, 0.5), (12, 1, 2, tc(2)), (20, 4, 2, 5.0)])
def test_seam_solve_reproduces_global_labels(oracle, L, G, q, T):
    from paper_1202_0635_b200 import stripes
    seed = 0x5EED0300 + L
    s = oracle.init_spins(L, q, seed)
    for t in range(3):
        bonds = oracle.bonds(L, q, POTTS, T, seed, t, s)
        want = oracle.label(L, bonds)
        rows = L // G
        local = [_stripe_local_labels(bonds, g * rows, rows, L) for g in range(G)]
        first = np.stack([l[0] for l in local])
        last = np.stack([l[-1] for l in local])
        seam = np.stack([(bonds[(g + 1) * rows - 1] >> 1) & 1 for g in range(G)]).astype(np.uint8)
        frm, to = stripes.solve_seams(first, last, seam)
        assert np.all(to < frm) and len(set(frm.tolist())) == len(frm)         # roots only move to smaller indices, one entry per root
        got = np.concatenate([_apply(l, frm, to) for l in local])
        assert np.array_equal(got, want), f"sweep {t}: global labels differ"
        s = oracle.sweep(L, q, POTTS, T, seed, t, s)


def _free_port():
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        return sk.getsockname()[1]


def _gloo_worker(rank, world, port, L, q, T, seed, ret):
    import torch.distributed as dist
    from oracle import sw_oracle as oracle
    from paper_1202_0635_b200 import stripes
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        rows = L // world
        s = oracle.init_spins(L, q, seed)
        ok = True
        for t in range(3):
            # every rank knows the whole configuration here only to cut its own stripe out of the oracle's bonds
            bonds = oracle.bonds(L, q, POTTS, T, seed, t, s)
            local = _stripe_local_labels(bonds, rank * rows, rows, L)
            seam = ((bonds[(rank + 1) * rows - 1] >> 1) & 1).astype(np.uint8)
            first = stripes.gather_rows(local[0], dist)
            last = stripes.gather_rows(local[-1], dist)
            seams = stripes.gather_rows(seam, dist)
            frm, to = stripes.solve_seams(first, last, seams)
            got = _apply(local, frm, to)
            want = oracle.label(L, bonds)[rank * rows:(rank + 1) * rows]
            ok = ok and bool(np.array_equal(got, want))
            s = oracle.sweep(L, q, POTTS, T, seed, t, s)
        ret[rank] = ok
    finally:
        dist.destroy_process_group()


def test_two_ranks_over_gloo_reproduce_the_oracle_labels(oracle):
    """world_size 2, gloo, CPU: each rank labels its half, the two all-gathers and the redundant seam solve give every
    rank the oracle's global labels on its rows."""
    import torch.multiprocessing as mp
    L, q, T, seed = 32, 2, tc(2), 0x5EED0301
    port = _free_port()
    with mp.Manager() as mgr:
        ret = mgr.dict()
        mp.spawn(_gloo_worker, args=(2, port, L, q, T, seed, ret), nprocs=2, join=True)
        assert ret.get(0) is True and ret.get(1) is True


@pytest.mark.gpu
@pytest.mark.parametrize("L,G,q,model,T", [(64, 2, 2, POTTS, tc(2)), (128, 4, 3, POTTS, tc(3)), (96, 8, 6, CLOCK, 0.9), (256, 2, 2, POTTS, 0.8 * tc(2)),
                                            (32, 1, 2, POTTS, tc(2)), (64, 16, 2, POTTS, 0.02)])
def test_stripes_on_one_gpu_equal_the_oracle(oracle, L, G, q, model, T):
    """G stripes of one lattice, held by one process and run one after the other: spins and canonical labels of every sweep
    equal the single-lattice oracle's."""
    from paper_1202_0635_b200 import stripes
    seed = 0x5EED0302 + L
    parts = [stripes.Stripe(L, q, model, T, seed, g, G) for g in range(G)]
    try:
        s = oracle.init_spins(L, q, seed)
        assert np.array_equal(np.concatenate([p.get_spins() for p in parts]), s), "S^0 differs"
        for t in range(4):
            stripes.sweep_local(parts)
            s, lab = oracle.sweep(L, q, model, T, seed, t, s, want_labels=True)
            assert np.array_equal(np.concatenate([p.get_labels() for p in parts]), lab), f"labels of sweep {t}"
            assert np.array_equal(np.concatenate([p.get_spins() for p in parts]), s), f"spins after sweep {t}"
        # hand-off at an absolute sweep index
        from paper_1202_0635_b200.workloads import random_spins
        s = random_spins(L, q, 9)
        rows = L // G
        for g, p in enumerate(parts):
            p.set_spins(s[g * rows:(g + 1) * rows], 17)
        stripes.sweep_local(parts)
        assert np.array_equal(np.concatenate([p.get_spins() for p in parts]), oracle.sweep(L, q, model, T, seed, 17, s))
    finally:
        for p in parts:
            p.close()
