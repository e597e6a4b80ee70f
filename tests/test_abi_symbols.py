"""CPU-side checks of the boundary: libspin.so builds (nvcc cross-compiles), loads, and exports every symbol
include/spin.h declares; argument validation that needs no GPU.  No compute calls here."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def P():
    import paper_1107_5463_b200 as pkg

    pkg.lib()
    return pkg


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "spin.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(spin_[a-z_]+)\s*\(", text)))


def test_header_symbols_are_exported(P):
    from paper_1107_5463_b200 import binding

    declared = _declared_symbols()
    assert len(declared) >= 15
    L = C.CDLL(binding.lib_path())
    for name in declared:
        assert hasattr(L, name), "libspin.so does not export %s" % name
    assert sorted(binding.SYMBOLS) == declared, "binding.SYMBOLS and include/spin.h disagree"
    assert b"sm_100a" in P.lib().spin_version()


def test_library_embeds_sm100a_code_only():
    from paper_1107_5463_b200 import binding, build

    out = os.popen("cuobjdump -lelf %s 2>/dev/null" % binding.lib_path()).read()
    if not out.strip():
        pytest.skip("cuobjdump unavailable")
    assert "sm_100a" in out
    assert "compute_100a" in " ".join(build.NVCC_FLAGS)
    assert "--use_fast_math" not in build.NVCC_FLAGS


def test_workspace_bytes_and_validation_without_gpu(P):
    cfg, _ = P.make_config((64, 64, 1), n=1, storage="int8")
    assert P.workspace_bytes(cfg) >= 4096
    cfg, _ = P.make_config((16384, 16384, 1), n=1, storage="bitpack")
    assert 33554432 <= P.workspace_bytes(cfg) < 34000000
    cfg, _ = P.make_config((16384, 16384, 1), n=1, storage="int8")
    assert 4 * 134217728 <= P.workspace_bytes(cfg) < 4 * 134217728 + 1000000   # two pairs of colour arrays (temporal blocking)
    cfg, _ = P.make_config((256, 256, 256), n=3, storage="fp32")
    assert P.workspace_bytes(cfg) >= 201326592
    cfg, _ = P.make_config((256, 256, 256), n=1, storage="bitpack", coupling="bond_pm1", replicas=16)
    assert P.workspace_bytes(cfg) >= 33554432 + 100663296
    bad = [
        dict(dims=(63, 64, 1)), dict(dims=(64, 64, 3)), dict(dims=(0, 4, 1)), dict(dims=(4, 4, 1), n=4),
        dict(dims=(4, 4, 1), n=1, storage="fp32"), dict(dims=(4, 4, 1), n=3, storage="int8"),
        dict(dims=(4, 4, 1), replicas=0),
    ]
    for kw in bad:
        cfg, _ = P.make_config(**kw)
        with pytest.raises(P.SpinError) as e:
            P.workspace_bytes(cfg)
        assert e.value.status == 1, kw
    unsupported = [
        dict(dims=(32, 32, 1), storage="bitpack"), dict(dims=(64, 64, 1), J=(0.5, 0.5, 0.5)),
        dict(dims=(64, 64, 1), n=3, storage="fp32", coupling="bond_pm1"),
        dict(dims=(64, 64, 1), storage="bitpack", coupling="per_direction"),
    ]
    for kw in unsupported:
        cfg, _ = P.make_config(**kw)
        with pytest.raises(P.SpinError) as e:
            P.workspace_bytes(cfg)
        assert e.value.status == 2, kw


def test_no_cpu_fallback(P):
    """Without a CUDA device the product path must fail loudly, not route through the oracle."""
    import torch

    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(RuntimeError):
        P.SpinSystem((64, 64, 1))
    src = open(os.path.join(ROOT, "paper_1107_5463_b200", "binding.py")).read()
    assert "oracle" not in src.replace("no CPU fallback", "")
