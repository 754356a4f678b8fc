"""Writes tests/golden/tiny_moe.json: a hand-derived worked example of the skip-token MoE layer.

The paper prints no numeric example of the layer, so this fixture is the closed form of PAPER.md Eq. 13, 14, 17
(+ the skip rule of PAPER.md:157-159 / 147 and BASELINE.json's SwiGLU expert) on inputs chosen so every quantity is
a rational multiple of ln2 / ln3.  This script only evaluates those hand-derived expressions with math.log; it
calls neither oracle/ nor the CUDA path.  Run: python tests/golden/make_tiny_moe.py
"""
import json
import math
from pathlib import Path

l2, l3 = math.log(2), math.log(3)
da = -0.75 * (1 + 0.25 * l3)
du = -0.375 * l3
dz = (0.125 * l3, 0.25 * l3, -0.375 * l3)
g = {
    "citation": "Layer definition PAPER.md:515 (Eq. 13), 519 (Eq. 14), 595 (Eq. 17), skip rule PAPER.md:157-159 + 147 (Fig. 3), expert PAPER.md:589 with BASELINE.json's SwiGLU form. The paper prints no numeric example; these values are closed forms derived by hand from those equations (derivation below), not produced by any implementation.",
    "derivation": [
        "T=1 token x=(1,2); d=2, E=3, k=2, F=1; resident S={0,2}; dy=(1,1).",
        "W_r=[[0,ln2,0],[0,0,ln3/2]] => z = x W_r = (0, ln2, ln3); softmax: e^z=(1,2,3) => p=(1/6,1/3,1/2); sigmoid: p=(1/2,2/3,3/4).",
        "top-2 by z: experts (2,1). Expert 1 is a ghost (not in S) => pair j=1 skipped, gate 0, no row. Expert 2 = slot 1.",
        "slot 1: W_g=(ln3,0) => a=ln3, sigmoid(a)=3/4, silu(a)=(3/4)ln3; W_u=(0,1) => u=2; h=(3/2)ln3; W_d=(1,-2)^T => o=((3/2)ln3, -3 ln3).",
        "softmax drop-only: g=1/2 => y=(3/4 ln3, -3/2 ln3). renorm_topk: g=(1/2)/(5/6)=3/5. renorm_resident: g=1. sigmoid drop-only: g=3/4.",
        "backward (softmax, drop-only): dg=<dy,o>=-(3/2)ln3; do=g dy=(1/2,1/2); dh=W_d^T do=-1/2;",
        "  da=dh u s(1+a(1-s))=-(3/4)(1+ln3/4); du=dh a s=-(3/8)ln3; dW_g=da x; dW_u=du x; dW_d=do h=(3/4 ln3, 3/4 ln3);",
        "  dp=(0,0,dg); sum_j p_j dp_j=-(3/4)ln3; dz_e=p_e(dp_e+(3/4)ln3) = (ln3/8, ln3/4, -(3/8)ln3); dW_r[i,e]=x_i dz_e;",
        "  dx = da W_g + du W_u + W_r dz = (da ln3 + ln2 ln3/4, du - (3/16) ln3^2).",
    ],
    "inputs": {"x": [[1.0, 2.0]], "dy": [[1.0, 1.0]], "w_router": [[0.0, l2, 0.0], [0.0, 0.0, l3 / 2]], "resident": [0, 2], "k": 2,
               "w_gate": [[[0.3, -0.2]], [[l3, 0.0]]], "w_up": [[[0.1, 0.4]], [[0.0, 1.0]]],
               "w_down": [[[0.5], [0.25]], [[1.0], [-2.0]]]},
    "expected": {
        "topk_idx": [[2, 1]], "pair_row": [[0, -1]], "counts": [0, 1], "offsets": [0, 0, 1], "row_token": [0],
        "probs_softmax": [[1 / 6, 1 / 3, 1 / 2]], "probs_sigmoid": [[0.5, 2 / 3, 0.75]],
        "gate_softmax_drop": [[0.5, 0.0]], "gate_softmax_renorm_topk": [[0.6, 0.0]],
        "gate_softmax_renorm_resident": [[1.0, 0.0]], "gate_sigmoid_drop": [[0.75, 0.0]],
        "y_softmax_drop": [[0.75 * l3, -1.5 * l3]], "y_sigmoid_drop": [[1.125 * l3, -2.25 * l3]],
        "y_softmax_renorm_topk": [[0.9 * l3, -1.8 * l3]], "y_softmax_renorm_resident": [[1.5 * l3, -3 * l3]],
        "bwd_softmax_drop": {
            "dgate": [[-1.5 * l3, 0.0]],
            "dlogits": [list(dz)],
            "dw_router": [[dz[0], dz[1], dz[2]], [2 * dz[0], 2 * dz[1], 2 * dz[2]]],
            "dw_gate": [[[0.0, 0.0]], [[da, 2 * da]]], "dw_up": [[[0.0, 0.0]], [[du, 2 * du]]],
            "dw_down": [[[0.0], [0.0]], [[0.75 * l3], [0.75 * l3]]],
            "dx": [[da * l3 + l2 * dz[1], du + (l3 / 2) * dz[2]]],
        },
    },
}
json.dump(g, open(Path(__file__).with_name("tiny_moe.json"), "w"), indent=1)
