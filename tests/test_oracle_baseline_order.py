"""Pins of oracle/baseline_order.py (Eqs. 1-2) against what the mathematics fixes."""
import itertools

import numpy as np

from oracle import baseline_order as bo


def test_eq1_worked_example_four_antennas():
    # upper triangle incl. the diagonal, numbered row by row (by hand): N_ant = 4
    expect = {(0, 0): 0, (0, 1): 1, (0, 2): 2, (0, 3): 3, (1, 1): 4, (1, 2): 5, (1, 3): 6, (2, 2): 7, (2, 3): 8, (3, 3): 9}
    for (a, b), k in expect.items():
        assert bo.baseline_index([a], [b], 4)[0] == k
        assert bo.baseline_index([b], [a], 4)[0] == k          # antenna order does not matter


def test_eq1_is_a_bijection_onto_the_triangle():
    for n in (1, 2, 3, 7, 64, 257):
        pairs = [(a, b) for a in range(n) for b in range(a, n)]
        ib = bo.baseline_index([p[0] for p in pairs], [p[1] for p in pairs], n)
        assert sorted(ib.tolist()) == list(range(bo.n_baseline_slots(n)))
        # row S of the triangle starts at S N - S (S - 1) / 2 (closed form of the quadratic term of Eq. 1)
        for S in range(n):
            assert bo.baseline_index([S], [S], n)[0] == S * n - S * (S - 1) // 2
        # lexicographic order of (min, max) is the order of I_B
        assert np.all(np.diff(ib) == 1)


def test_eq2_is_the_exclusive_prefix_sum_and_reorder_is_stable():
    rng = np.random.default_rng(7)
    n_ant, nrow = 9, 5000
    a1 = rng.integers(0, n_ant, nrow); a2 = rng.integers(0, n_ant, nrow)
    C, B = bo.start_index(a1, a2, n_ant)
    ib = bo.baseline_index(a1, a2, n_ant)
    assert C.sum() == nrow and B[0] == 0 and B[-1] == nrow
    assert np.array_equal(C, np.bincount(ib, minlength=bo.n_baseline_slots(n_ant)))
    assert np.array_equal(B[1:], np.cumsum(C))                  # library routine
    perm = bo.reorder(a1, a2, n_ant)
    assert sorted(perm.tolist()) == list(range(nrow))
    assert np.array_equal(perm, np.argsort(ib, kind="stable"))   # grouped by baseline, time order kept
    for k in range(bo.n_baseline_slots(n_ant)):
        seg = perm[B[k]:B[k + 1]]
        assert np.all(ib[seg] == k) and np.all(np.diff(seg) > 0)


def test_time_major_data_gives_one_row_per_dump_per_baseline():
    n_ant, n_dump = 6, 11
    i, j = np.triu_indices(n_ant, k=1)
    a1 = np.tile(i, n_dump); a2 = np.tile(j, n_dump)
    C, B = bo.start_index(a1, a2, n_ant)
    ib_cross = bo.baseline_index(i, j, n_ant)
    assert np.all(C[ib_cross] == n_dump) and C.sum() == n_dump * i.size       # autocorrelation slots stay empty
    perm = bo.reorder(a1, a2, n_ant)
    nbl = i.size
    for b, k in enumerate(ib_cross):
        assert np.array_equal(perm[B[k]:B[k + 1]], b + nbl * np.arange(n_dump))
