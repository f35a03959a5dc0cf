"""The overflow paths of the tile kernel (union-edge list, root list) are unreachable with the production list
capacities on the paper's workloads; this test builds the same library with tiny capacities (SW_EDGE_CAP=8,
SW_RCAP=16, SW_NARROW_MAX=40: tiles with more open roots write two bytes per site) so that every warp overflows both lists and both label formats occur, and checks parity with the oracle, bit for bit."""
import os
import subprocess
import sys
from pathlib import Path

import pytest

pytestmark = pytest.mark.gpu
ROOT = Path(__file__).resolve().parents[1]

SCRIPT = r"""
import math, sys
import numpy as np
sys.path.insert(0, %r)
from oracle import sw_oracle as o
from paper_1202_0635_b200 import binding as sw
tc2 = 1.0 / math.log(1.0 + math.sqrt(2.0))
for (L, q, model, T) in ((256, 2, 0, tc2), (256, 6, 1, 0.9), (128, 2, 0, 1e6), (256, 3, 0, 0.3)):
    seed = 0x5EED0077
    with sw.Lattice(L, q, model, T, seed, algo=sw.SW_ALGO_TILED) as lat:
        s = o.init_spins(L, q, seed)
        for t in range(4):
            lat.sweep(1)
            s, lab = o.sweep(L, q, model, T, seed, t, s, want_labels=True)
            assert np.array_equal(lat.get_labels(), lab), (L, q, model, T, t, "labels")
            assert np.array_equal(lat.get_spins(), s), (L, q, model, T, t, "spins")
print("overflow parity ok")
"""


def test_tiny_list_capacities_match_the_oracle(tmp_path):
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1202_0635_b200 import build
    lib = tmp_path / "libsw_tiny.so"
    cmd = [os.environ.get("NVCC", "nvcc"), *build.NVCC_FLAGS, "-DSW_EDGE_CAP=8", "-DSW_RCAP=16", "-DSW_NARROW_MAX=40",
           "-I", str(ROOT / "include"), "-I", str(build.CSRC), "-o", str(lib)] + [str(s) for s in build.sources()]
    subprocess.run(cmd, check=True)
    env = dict(os.environ, SW_LIB=str(lib))
    out = subprocess.run([sys.executable, "-c", SCRIPT % str(ROOT)], env=env, capture_output=True, text=True, timeout=600)
    assert out.returncode == 0, out.stdout + out.stderr
    assert "overflow parity ok" in out.stdout
