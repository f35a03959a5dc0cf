"""sw_sweep_noalloc (include/sw.h): the sweep whose scratch is a static device array of libsw.so, for callers that
cannot call cudaMalloc.  Its output is compared bit for bit (the bar of tests/test_gpu_parity.py) with the existing
path's -- a context made by sw_create_in, any back-end -- on two calls in a row and across problems of different
size that reuse the one scratch array.

This file is named so that pytest collects it last (the run uses -x).
"""
from __future__ import annotations

import math

import numpy as np
import pytest

POTTS, CLOCK = 0, 1
GENERIC = 1


def tc(q):
    return 1.0 / math.log(1.0 + math.sqrt(float(q)))


@pytest.fixture(scope="module")
def sw():
    from paper_1202_0635_b200 import build, binding
    build.build()
    binding.load()
    return binding


def _existing_path(sw, L, q, model, T, seed, n, algo=0):
    """S^0 .. S^n of the existing path (a context, default back-end for this L unless `algo` is given)."""
    out = []
    with sw.Lattice(L, q, model, T, seed, algo=algo) as lat:
        out.append(lat.get_spins().copy())
        for _ in range(n):
            lat.sweep(1)
            out.append(lat.get_spins().copy())
    return out


def _assert_same(a, b, what):
    if not np.array_equal(a, b):
        bad = np.argwhere(np.asarray(a) != np.asarray(b))
        raise AssertionError(f"{what}: {len(bad)} mismatches, first at {bad[:5].tolist()}")


CASES = [
    # L, q, model, T factor (of the Potts T_c, or absolute for the clock model), seed
    (512, 2, POTTS, 1.0, 11),        # tiled back-end on the existing side
    (1024, 3, POTTS, 1.0, 12),       # the maximum size
    (256, 6, CLOCK, None, 13),       # clock model: threshold table in the scratch
    (67, 5, POTTS, 0.9, 14),         # odd L, large clusters, generic back-end on the existing side
    (48, 4, CLOCK, None, 15),        # one-CTA back-end on the existing side
]


@pytest.mark.gpu
@pytest.mark.parametrize("L,q,model,tf,seed", CASES)
def test_noalloc_sweep_equals_existing_path_on_consecutive_calls(sw, L, q, model, tf, seed):
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    T = tc(q) * tf if model == POTTS else 0.9
    ref = _existing_path(sw, L, q, model, T, seed, 3)
    d = [torch.from_numpy(ref[0]).cuda(), torch.empty((L, L), dtype=torch.uint8, device="cuda"),
         torch.empty((L, L), dtype=torch.uint8, device="cuda")]
    # two calls in a row, no synchronisation between them: the second reads what the first wrote, both use the scratch
    sw.sweep_noalloc(L, q, model, T, seed, 0, d[0], d[1])
    sw.sweep_noalloc(L, q, model, T, seed, 1, d[1], d[2])
    torch.cuda.synchronize()
    _assert_same(d[1].cpu().numpy(), ref[1], "first call (sweep 0)")
    _assert_same(d[2].cpu().numpy(), ref[2], "second call (sweep 1)")
    # third call in place (in == out)
    sw.sweep_noalloc(L, q, model, T, seed, 2, d[2], d[2])
    torch.cuda.synchronize()
    _assert_same(d[2].cpu().numpy(), ref[3], "third call, in place (sweep 2)")
    _assert_same(d[0].cpu().numpy(), ref[0], "the input buffer of the first call is untouched")


@pytest.mark.gpu
def test_noalloc_scratch_is_shared_and_stale_contents_do_not_leak(sw):
    """Problems of different size and model alternate on the one scratch array; every result still equals the
    existing path's, and the device's free memory does not move (nothing is allocated)."""
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    probs = [(1024, 2, POTTS, tc(2), 21), (96, 8, CLOCK, 0.7, 22), (333, 3, POTTS, tc(3) * 0.95, 23), (128, 6, CLOCK, 1.1, 24)]
    ref = [_existing_path(sw, L, q, m, T, seed, 2, algo=GENERIC) for (L, q, m, T, seed) in probs]
    bufs = [(torch.from_numpy(r[0]).cuda(), torch.empty(r[0].shape, dtype=torch.uint8, device="cuda"),
             torch.empty(r[0].shape, dtype=torch.uint8, device="cuda")) for r in ref]
    for (L, q, m, T, seed), b in zip(probs, bufs):   # first use of every kernel (lazy module loading happens here)
        sw.sweep_noalloc(L, q, m, T, seed, 0, b[0], b[1])
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for rep in range(3):
        for (L, q, m, T, seed), b in zip(probs, bufs):
            sw.sweep_noalloc(L, q, m, T, seed, 0, b[0], b[1])
            sw.sweep_noalloc(L, q, m, T, seed, 1, b[1], b[2])
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free0 - free1 < (1 << 20), f"device free memory fell by {free0 - free1} bytes over 24 calls"
    for (L, q, m, T, seed), b, r in zip(probs, bufs, ref):
        _assert_same(b[1].cpu().numpy(), r[1], f"L={L} q={q} model={m}: sweep 0")
        _assert_same(b[2].cpu().numpy(), r[2], f"L={L} q={q} model={m}: sweep 1")


@pytest.mark.gpu
def test_noalloc_rejects_what_it_cannot_serve(sw):
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    L = 64
    a = torch.zeros((L, L), dtype=torch.uint8, device="cuda")
    host = np.zeros((L, L), dtype=np.uint8)
    with pytest.raises(sw.SwError) as e:
        sw.sweep_noalloc(L, 2, POTTS, 1.0, 1, 0, host.ctypes.data, a)     # a host pointer
    assert e.value.code == sw.SW_ERR_ARG and "device memory" in str(e.value)
    with pytest.raises(sw.SwError) as e:
        sw.sweep_noalloc(L, 2, POTTS, 1.0, 1, 0, a.data_ptr(), a.data_ptr() + 16)   # partial overlap
    assert e.value.code == sw.SW_ERR_ARG and "overlap" in str(e.value)
    with pytest.raises(sw.SwError) as e:
        sw.sweep_noalloc(L, 2, POTTS, 1.0, 1, 1 << 32, a, a)
    assert e.value.code == sw.SW_ERR_ARG
    torch.cuda.synchronize()
    assert int(a.sum().item()) == 0, "a rejected call enqueued work"


def test_noalloc_size_limit_is_checked_before_any_cuda_call(sw):
    """No GPU needed: sizes beyond the static scratch are refused with a message that names the limit."""
    lib = sw.load()
    assert sw.SW_NOALLOC_MAX_L == 1024
    rc = lib.sw_sweep_noalloc(sw.SW_NOALLOC_MAX_L + 1, 2, POTTS, 1.0, 1, 0, None, None, None)
    assert rc == sw.SW_ERR_UNSUPPORTED
    msg = sw.last_error()
    assert "SW_NOALLOC_MAX_L = 1024" in msg and "1025" in msg
    assert lib.sw_sweep_noalloc(4096, 2, POTTS, 1.0, 1, 0, None, None, None) == sw.SW_ERR_UNSUPPORTED
    for bad in [(1, 2, POTTS, 1.0), (64, 1, POTTS, 1.0), (64, 17, POTTS, 1.0), (64, 2, 2, 1.0), (64, 2, POTTS, 0.0),
                (64, 2, POTTS, float("nan"))]:
        assert lib.sw_sweep_noalloc(bad[0], bad[1], bad[2], bad[3], 1, 0, None, None, None) == sw.SW_ERR_ARG
    assert lib.sw_sweep_noalloc(64, 2, POTTS, 1.0, 1, 0, None, None, None) == sw.SW_ERR_ARG   # NULL buffers
    assert "NULL" in sw.last_error()
