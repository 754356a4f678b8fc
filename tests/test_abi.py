"""Host-side checks of the C-ABI library that need no GPU: it loads, exports every symbol include/fomoe.h declares,
and its host-only entry points (argument checks, workspace sizing) behave."""
import ctypes as C
import re
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parents[1]


@pytest.fixture(scope="module")
def B():
    from paper_2606_19025_b200 import build
    build.build()
    from paper_2606_19025_b200 import binding
    binding.lib()
    return binding


def test_exports_match_header(B):
    header = (ROOT / "include" / "fomoe.h").read_text()
    declared = set(re.findall(r"FOMOE_API\s+[\w\s\*]+?\b(fomoe_\w+)\s*\(", header))
    assert declared and declared == set(B.EXPORTS)
    lib = C.CDLL(str(B.LIB_PATH))
    for name in declared:
        assert hasattr(lib, name), name
    assert lib.fomoe_abi_version() == 5


def test_workspace_sizes_and_argument_checks(B):
    cfg = B.make_config(T=8192, d_model=1024, E=16, top_k=2, d_ff=2816)
    r, a, s = B.fomoe_workspace_bytes(cfg, 8)
    rows = (8192 * 2 + 127) // 128 * 128 + 8 * 128
    assert a >= rows * (2 * 1024 + 3 * 2816) * 2            # xp, o, a, u, h in bf16 for the worst-case padded rows
    assert r >= rows * 12 and s >= rows * (2 * 1024 + 2 * 2816) * 2
    for bad in (dict(top_k=17), dict(T=-1), dict(d_model=0), dict(dtype=7), dict(temperature=0.0), dict(gate_rule=3)):
        kw = dict(T=16, d_model=64, E=16, top_k=2, d_ff=64)
        kw.update(bad)
        with pytest.raises(B.FomoeError, match="BADARG"):
            B.fomoe_workspace_bytes(B.make_config(**kw), 4)
    with pytest.raises(B.FomoeError, match="UNSUPPORTED"):
        B.fomoe_workspace_bytes(B.make_config(T=16, d_model=64, E=1024, top_k=2, d_ff=64), 4)
    with pytest.raises(B.FomoeError, match="BADARG"):
        B.fomoe_workspace_bytes(cfg, 17)


def test_product_path_fails_loudly_without_gpu(B):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    from paper_2606_19025_b200 import workloads as W
    from paper_2606_19025_b200.layer import SkipTokenMoE
    w = W.config("C1")
    S = W.resident_set(w)
    with pytest.raises(B.FomoeError):
        SkipTokenMoE(w, S, W.make_router(w), *W.make_resident_experts(w, S))


def test_product_does_not_import_oracle():
    for f in (ROOT / "paper_2606_19025_b200").rglob("*.py"):
        src = f.read_text()
        assert "oracle" not in src.replace("oracle's", ""), f
    for f in (ROOT / "oracle").glob("*.py"):
        assert "paper_2606_19025_b200" not in f.read_text(), f
