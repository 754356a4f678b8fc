"""Pins for oracle/stats_oracle.py: closed forms the definitions fix (Eq. 2)."""
import numpy as np

from oracle import stats_oracle as SO


def test_perfectly_balanced_load():
    """Every expert gets the same number of assignments: CV = 0, entropy = ln E, kept fraction = N_le / N_e (Eq. 2)."""
    E, k, reps = 8, 2, 5
    idx = np.array([[(2 * t) % E, (2 * t + 1) % E] for t in range(reps * E // 2)], np.int32)
    s = SO.routing_stats(idx, np.arange(E // 2, dtype=np.int32), E)
    assert np.all(s["load"] == reps)
    assert abs(s["load_cv"]) < 1e-15 and abs(s["routing_entropy"] - np.log(E)) < 1e-12
    assert abs(s["kept_fraction"] - 0.5) < 1e-15 and abs(s["ghost_fraction"] - 0.5) < 1e-15
    # pairs (0,1), (2,3) kept entirely, (4,5), (6,7) ghost entirely
    assert abs(s["zero_kept_tokens"] - 0.5) < 1e-15


def test_collapsed_router():
    """All tokens pick expert 3 (k = 1): entropy 0, CV = sqrt(E - 1) (one-hot load), everything kept iff 3 is resident."""
    E, T = 16, 40
    idx = np.full((T, 1), 3, np.int32)
    s = SO.routing_stats(idx, np.array([3], np.int32), E)
    assert s["routing_entropy"] == 0.0 and abs(s["load_cv"] - np.sqrt(E - 1)) < 1e-12
    assert s["kept_fraction"] == 1.0 and s["zero_kept_tokens"] == 0.0 and s["max_load"] == T and s["min_load"] == 0
    s = SO.routing_stats(idx, np.array([4, 5], np.int32), E)
    assert s["kept_fraction"] == 0.0 and s["ghost_fraction"] == 1.0 and s["zero_kept_tokens"] == 1.0


def test_two_level_load_closed_form():
    """Half of the experts carry 3 assignments, half carry 1: mean 2, std 1 -> CV 1/2; entropy from the two frequencies."""
    E = 4
    idx = np.array([[0], [0], [0], [1], [1], [1], [2], [3]], np.int32)
    s = SO.routing_stats(idx, np.array([0, 2], np.int32), E)
    assert abs(s["load_cv"] - 0.5) < 1e-15
    want = -(2 * (3 / 8) * np.log(3 / 8) + 2 * (1 / 8) * np.log(1 / 8))
    assert abs(s["routing_entropy"] - want) < 1e-12
    assert abs(s["kept_fraction"] - 4 / 8) < 1e-15
