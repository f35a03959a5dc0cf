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
    return sorted(set(re.findall(r"\b(sw_[A-Za-z0-9_]+)\s*\(", text)))


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


def test_derived_doubles_are_host_functions_with_closed_forms(lib):
    """sw_derive_* (eq.(2), (3), (5), (6)) need no device: closed forms and argument errors.  (Their comparison
    with the oracle's own functions is a -m gpu test over recorded series, tests/test_gpu_parity.py.)"""
    import math
    import numpy as np
    from paper_1202_0635_b200 import binding as sw
    N = 64 * 64
    assert sw.potts_energy(64, [2 * N, 0]) == 0.0 and sw.potts_energy(64, [0, 2 * N]) == 2.0 * N
    assert sw.potts_m2(2, [N, 0]) == float(N * N) and sw.potts_m2(2, [N // 2, N // 2]) == 0.0       # uniform / half-half
    assert sw.potts_m2(3, [0, N, 0]) == float(N * N) and sw.potts_m2(16, [1 << 28] + [0] * 15) == float(1 << 56)
    assert sw.clock_energy(6, [2 * N, 0, 0, 0, 0, 0]) == -2.0 * N
    assert abs(sw.clock_m(6, [N, 0, 0, 0, 0, 0]) - N) < 1e-9 and sw.clock_m(6, [5, 0, 0, 5, 0, 0]) < 1e-9
    assert sw.g(2, [0, 32]) == -1.0 and sw.g(6, [7, 0, 0, 0, 0, 0]) == 1.0                          # checkerboard odd r / uniform
    assert sw.moment_ratio(2, [[N, 0]] * 3) == 1.0
    assert abs(sw.moment_ratio(2, [[1, 0], [4, 0]]) - (257.0 / 2.0) / (8.5 * 8.5)) < 1e-15
    assert abs(sw.ratio_R(2, [[3, 1], [2, 2]], [[4, 0], [3, 1]]) - 0.25 / 0.75) < 1e-15
    assert sw.ratio_R(6, [[9, 0, 0, 0, 0, 0]], [[9, 0, 0, 0, 0, 0]]) == 1.0
    assert math.isnan(lib.sw_derive_potts_m2(1, np.zeros(2, dtype=np.int64).ctypes.data))
    assert math.isnan(lib.sw_derive_g(6, None)) and math.isnan(lib.sw_derive_moment_ratio(0, 2, np.zeros(2, dtype=np.int64).ctypes.data))


def test_binding_holds_no_arithmetic_of_the_method():
    """binding.py marshals; the doubles come from libsw.so (derived observables out of the binding)."""
    txt = (ROOT / "paper_1202_0635_b200" / "binding.py").read_text()
    for token in ("math.cos", "math.sin", "math.hypot", "import math", "np.cos", "np.exp"):
        assert token not in txt, token


def test_pdl_kernels_never_read_producer_buffers_through_nc_loads(lib):
    """a kernel of the programmatic-dependent-launch chain must not load a buffer the previous kernel writes
    with ld.global.nc (LDG.E.CONSTANT), and no global load may precede griddepcontrol.wait (ACQBULK).  Read off the SASS."""
    import shutil
    import subprocess
    from paper_1202_0635_b200 import binding
    if not shutil.which("cuobjdump"):
        pytest.skip("cuobjdump not on PATH")
    sass = subprocess.run(["cuobjdump", "-sass", str(binding.LIB_PATH)], capture_output=True, text=True, check=True).stdout
    seen = 0
    for f in re.split(r"\n\s*Function : ", sass)[1:]:
        name = f.split("\n")[0]
        if not any(k in name for k in ("k_tile_label", "k_seam_merge", "k_tile_flip", "k_observables", "k_correlation")):
            continue
        seen += 1
        lines = [l for l in f.split("\n") if re.match(r"\s*/\*[0-9a-f]{4}\*/", l)]
        acq = next((i for i, l in enumerate(lines) if "ACQBULK" in l), None)
        assert acq is not None, f"{name}: no griddepcontrol.wait"
        loads = [i for i, l in enumerate(lines) if re.search(r"\bLDG\b|\bLDG\.|\bLD\.E", l)]
        assert loads and min(loads) > acq, f"{name}: a global load precedes griddepcontrol.wait"
        assert not [l for l in lines if "LDG" in l and "CONSTANT" in l], f"{name}: ld.global.nc on a PDL kernel"
    assert seen >= 8


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
