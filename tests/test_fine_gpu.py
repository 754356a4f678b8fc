"""The gathered fine-grained expert kernels (csrc/fine_gemm.cu: d_expert = 128, d_model % 256 == 0, bf16, two-matrix expert;
PAPER.md:300-309, 589) against the fp64 oracle, element by element, through the C ABI: every output of the forward and the
backward.  The cases walk the kernel's schedule: only single row tiles (few pairs), full rounds of tile pairs plus a tail of
singles, slots with no token at all (zero weight gradients), one token, every expert resident, the split-K form of the
weight gradients (few output tiles) and its un-split form (many)."""
import os

import numpy as np
import pytest

import helpers as H
from paper_2606_19025_b200 import workloads as W
from test_parity_gpu import run_and_compare

pytestmark = pytest.mark.gpu


def _w(name, **kw):
    base = dict(T=900, d=256, E=16, k=4, F=128, n_res=8, gate_fn=W.GATE_SIGMOID, expert_fn=W.EXPERT_SILU, seed=11)
    base.update(kw)
    return W.MoEWorkload(name, **base)


def test_fine_path_is_the_one_that_runs():
    """The shapes below must take the gathered kernels: the library names its launches, and a forward + backward of such a
    shape launches fine_gather_kernel<F1 / DH / WG> and neither gather_rows nor scale_rows."""
    if os.environ.get("FOMOE_FINE", "7") != "7":
        pytest.skip("FOMOE_FINE overrides the default path")
    import torch
    from paper_2606_19025_b200 import binding as B
    p = H.Problem(_w("fine_names"))
    layer = H.make_layer(p)
    x, dy = layer.to_dev(p.x), layer.to_dev(p.dy)
    layer.step(x, dy)
    torch.cuda.synchronize()
    B.fomoe_profile_enable(True)
    layer.step(x, dy)
    names = {n for n, _ in B.fomoe_profile_collect(4096)}
    B.fomoe_profile_enable(False)
    assert {"fine_gather_kernel<F1>", "fine_gather_kernel<DH>", "fine_gather_kernel<WG>"} <= names, names
    assert not any(n.startswith(("gather_rows", "scale_rows", "combine_bwd")) for n in names), names


@pytest.mark.parametrize("kw", [
    dict(),                                            # 8 slots x ~450 rows: single tiles only, split-K weight gradients (16 tiles)
    dict(T=1, n_res=8),                                # one token: most slots empty -> zero dW rows, one live row per tile
    dict(T=3, k=2, n_res=8),                           # at most 6 pairs
    dict(T=127, n_res=3),
    dict(T=700, n_res=16),                             # every expert resident
    dict(T=1500, n_sh=1, F_sh=192, n_res=7),           # a shared expert beside the gathered routed path
    dict(T=640, d=1024, E=32, k=8, n_res=16, seed=12), # 16 x 2 x 4 = 128 weight-gradient tiles: one K part
    dict(T=500, d=1024, E=32, k=8, n_res=20, seed=14), # 160 tiles on 148 SMs: one full round stored directly, 12 tail tiles in 8 K parts
    dict(T=600, d=512, gate_fn=W.GATE_SOFTMAX, gate_rule=W.RULE_RENORM_RESIDENT),
], ids=lambda kw: "-".join(f"{k}{v}" for k, v in kw.items()) or "base")
def test_fine_full_parity(oracle64, kw):
    errs, _ = run_and_compare(H.Problem(_w("fine", **kw)), oracle64)
    print("fine", kw, errs)


def test_fine_many_pairs_full_rounds(oracle64):
    """More row-tile pairs than SMs: full rounds of pairs, then the tail handed out as single tiles (T = 12000, k = 8, half of
    the experts resident: ~48 k kept pairs = ~190 pairs over 148 CTAs)."""
    w = _w("fine_rounds", T=12000, d=256, E=16, k=8, n_res=8, seed=13)
    errs, _ = run_and_compare(H.Problem(w), oracle64)
    print("fine_rounds", errs)


@pytest.mark.parametrize("name", ["P1", "P2", "P3"])
def test_paper_shapes_full_size_every_element(oracle64, name):
    """The paper's Medium, Large and XL shapes at full size (P1: T = 16384, d_model = 512, 16 experts of width 128, 4 active, 8
    resident; P2: d_model = 1024, 32 experts, 8 active, 16 resident; P3: d_model = 2048, 64 experts, 16 active, 32 resident;
    PAPER.md:300-309), i.e. exactly what bench.py --workload P1|P2|P3 times: every element of every output of the
    forward and the backward against the fp64 oracle — 256 / 512 / 1048 row tiles (full rounds of pairs + the tail of singles),
    the split-K (P1), single-round (P2) and multi-round (P3) weight gradients, two token rows per CTA in combine / dx_sum (P1)."""
    errs, _ = run_and_compare(H.Problem(W.config(name)), oracle64)
    print(name, "full", errs)
