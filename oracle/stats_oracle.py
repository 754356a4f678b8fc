"""ORACLE — TEST INFRASTRUCTURE, NOT THE PRODUCT.  Routing diagnostics written out from their definitions (numpy, fp64).

The paper names them without formulas ("routing entropy, load coefficients of variation, and overflow rates";
PAPER.md:207 "the actual frequency of the token assignments to ghost experts against the total number of assignments"), so
each takes its textbook definition (reading R15):
  load[e]          number of (token, j) assignments with topk_idx[t,j] == e, over all E experts
  load CV          population standard deviation of load / mean of load
  routing entropy  Shannon entropy (nats) of the assignment distribution f_e = load[e] / (T k)
  ghost fraction   assignments to non-resident experts / all assignments;  kept fraction = 1 - that (sigma_st)
  zero-kept tokens fraction of tokens none of whose k selected experts is resident
Pinned in tests/test_oracle_stats.py (closed forms: balanced load, one-hot load, Eq. 2).  Imports nothing from the CUDA package.
"""
import numpy as np


def routing_stats(topk_idx: np.ndarray, resident: np.ndarray, E: int) -> dict:
    T, k = topk_idx.shape
    load = np.zeros(E, np.int64)
    for t in range(T):
        for j in range(k):
            load[topk_idx[t, j]] += 1
    total = float(T * k)
    mean = total / E
    cv = float(np.sqrt(((load - mean) ** 2).sum() / E) / mean) if total > 0 else 0.0
    f = load[load > 0] / total if total > 0 else np.zeros(0)
    ent = float(-(f * np.log(f)).sum())
    res = set(int(e) for e in resident)
    kept = np.array([[int(e) in res for e in row] for row in topk_idx], bool).reshape(T, k)
    kf = float(kept.sum() / total) if total > 0 else 0.0
    return dict(load=load, load_cv=cv, routing_entropy=ent, kept_fraction=kf, ghost_fraction=(1.0 - kf) if total > 0 else 0.0,
                zero_kept_tokens=float((~kept.any(1)).mean()) if T > 0 else 0.0, max_load=float(load.max()), min_load=float(load.min()))
