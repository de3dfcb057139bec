"""CPU-side checks of the C-ABI boundary: the library builds for sm_100a, loads, exports
every symbol include/tpcclus.h declares, sizes its workspace sanely and refuses to compute
without a CUDA device (no CPU fallback)."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def binding():
    from paper_2511_17018_b200 import build as b
    b.build()
    from paper_2511_17018_b200 import binding
    return binding


def test_exports_match_header(binding):
    hdr = open(os.path.join(ROOT, "include", "tpcclus.h")).read()
    declared = set(re.findall(r"TPCCLUS_API[^;(]*?\b(tpcclus_\w+)\s*\(", hdr))
    assert len(declared) >= 10 and {"tpcclus_create", "tpcclus_run", "tpcclus_destroy"} <= declared
    L = binding.lib()
    for name in declared:
        assert hasattr(L, name), name
    assert declared == set(binding.EXPORTS)


def test_record_sizes_match_header(binding):
    assert C.sizeof(binding.tpcclus_params) == 64 and C.sizeof(binding.tpcclus_out) == 32
    assert binding.DIGIT_DTYPE.itemsize == 8 and binding.CLUSTER_DTYPE.itemsize == 32


def test_workspace_bytes_and_validation(binding):
    from workloads import n_pads_ramp
    pads = n_pads_ramp(152)
    p, keep = binding.make_params(36, 152, 14256, pads, 1_590_000_000)
    w = binding.tpcclus_workspace_bytes(p)
    assert 10e9 < w < 16e9          # 13.4 GB at CFG[4]
    assert binding.tpcclus_workspace_bytes_host(p, 10**8) == pytest.approx(w + 8 * 1_590_000_000 + 32 * 10**8, rel=1e-6)
    small, keep2 = binding.make_params(1, 16, 256, [64] * 16, 10000)
    assert 0 < binding.tpcclus_workspace_bytes(small) < 200e6
    bad, _ = binding.make_params(0, 16, 256, [64] * 16, 10000)
    assert binding.tpcclus_workspace_bytes(bad) == 0
    bad, _ = binding.make_params(1, 16, 256, [64] * 15 + [300], 10000)
    assert binding.tpcclus_workspace_bytes(bad) == 0
    longer, keep3 = binding.make_params(36, 152, 40000, pads, 10**8)   # 16416 coarse bins: three passes of K1 (R1)
    assert binding.tpcclus_workspace_bytes(longer) > 0
    toomany, _ = binding.make_params(256, 256, 256, [64] * 256, 10000)   # 65536 coarse bins
    assert binding.tpcclus_workspace_bytes(toomany) == 0
    assert binding.lib().tpcclus_error_string(-5).startswith(b"unsupported")


def test_no_cpu_fallback(binding):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(RuntimeError):
        binding.Clusterizer(1, 16, 256, [64] * 16, 1000)
    # and the C entry point itself refuses: create needs a device
    buf = np.zeros(1 << 20, dtype=np.uint8)
    p, keep = binding.make_params(1, 1, 64, [16], 100)
    addr = (buf.ctypes.data + 255) & ~255
    p.workspace, p.workspace_bytes = addr, binding.tpcclus_workspace_bytes(p)
    with pytest.raises(binding.TpcclusError) as e:
        binding.tpcclus_create(p)
    assert e.value.code == -2
