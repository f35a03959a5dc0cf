"""CPU-only checks of the boundary: libsw.so loads and exports every symbol include/sw.h declares; argument
errors are reported without a GPU; no compute call is made."""
from __future__ import annotations

import ctypes
import re
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent


@pytest.fixture(scope="module")
def lib():
    from paper_1202_0635_b200 import build, binding
    build.build()
    return binding.load()


def _declared_symbols():
    text = (ROOT / "include" / "sw.h").read_text()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(sw_[a-z_]+)\s*\(", text)))


def test_header_symbols_exported_and_bound(lib):
    from paper_1202_0635_b200 import binding
    names = _declared_symbols()
    assert len(names) >= 20
    for n in names:
        assert hasattr(lib, n), f"libsw.so does not export {n}"
        assert n in binding.SYMBOLS, f"binding.py does not declare {n}"
    assert sorted(binding.SYMBOLS) == names


def test_workspace_bytes_and_argument_errors(lib):
    from paper_1202_0635_b200 import binding
    assert lib.sw_workspace_bytes(64, 2, 0) >= 64 * 64 * 6
    assert lib.sw_workspace_bytes(16384, 2, 0) >= 16384 * 16384 * 6
    assert lib.sw_workspace_bytes(1, 2, 0) == 0          # L < 2
    assert lib.sw_workspace_bytes(32768, 2, 0) == 0      # L > SW_MAX_L
    assert lib.sw_workspace_bytes(64, 1, 0) == 0         # q < 2
    assert lib.sw_workspace_bytes(64, 17, 0) == 0        # q > SW_MAX_Q
    assert lib.sw_workspace_bytes(64, 2, 2) == 0         # unknown model
    # argument validation happens before any CUDA call
    assert not lib.sw_create(1, 2, 0, 1.0, 1)
    assert b"sw_create" in lib.sw_last_error()
    assert not lib.sw_create(64, 2, 0, 0.0, 1)
    assert not lib.sw_create(64, 2, 0, float("nan"), 1)
    assert not lib.sw_create(64, 2, 0, float("inf"), 1)
    assert not lib.sw_create(64, 2, 5, 1.0, 1)
    # NULL contexts
    assert lib.sw_sweep(None, 1) == binding.SW_ERR_ARG
    assert lib.sw_sync(None) == binding.SW_ERR_ARG
    assert lib.sw_get_spins(None, None) == binding.SW_ERR_ARG
    assert lib.sw_observables(None, None, None) == binding.SW_ERR_ARG
    assert lib.sw_sweep_index(None) == 0
    assert lib.sw_launch_count(None) == 0
    lib.sw_destroy(None)


def test_no_cpu_fallback_without_gpu(lib):
    """Without a CUDA device creation fails loudly (SW_ERR_CUDA text), it never computes on the host."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    from paper_1202_0635_b200 import binding
    assert not lib.sw_create(64, 2, 0, 1.0, 1)
    assert b"no usable CUDA device" in lib.sw_last_error()
    with pytest.raises(binding.SwError):
        binding.Lattice(64, 2, 0, 1.0, 1)


def test_product_path_does_not_touch_the_oracle():
    """Nothing under the package imports, includes, loads or links oracle/ (and the oracle does not import the package)."""
    imp = re.compile(r"^\s*(from|import)\s+[^#\n]*oracle", re.M)
    inc = re.compile(r"#\s*include[^\n]*oracle")
    for p in (ROOT / "paper_1202_0635_b200").rglob("*"):
        if p.suffix in {".py", ".cu", ".cuh", ".h"}:
            txt = p.read_text()
            assert not imp.search(txt) and not inc.search(txt), p
            assert "libsw_oracle" not in txt and "sw_oracle.py" not in txt, p
    assert not inc.search((ROOT / "include" / "sw.h").read_text())
    for p in (ROOT / "oracle").rglob("*.py"):
        assert not re.search(r"^\s*(from|import)\s+[^#\n]*paper_1202_0635_b200", p.read_text(), re.M), p
    assert "#include \"sw" not in (ROOT / "oracle" / "sw_oracle.c").read_text()
