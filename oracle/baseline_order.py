"""Eqs. (1)-(2) of the paper — baseline index and baseline-then-time re-order (oracle, test infrastructure only).

PAPER.md:62-78 (§2.2): the CUDA gridder needs the data "grouped by baseline and then ordered by time".  The
Measurement Set stores only antenna IDs, so

    I_B = (-S^2 + 2 S N_ant + S) / 2 + |I_ant1 - I_ant2|,   S = min(I_ant1, I_ant2)        (Eq. 1)

numbers the baselines (autocorrelations included: row S of the upper triangle starts at
S N_ant - S (S - 1) / 2), the samples per baseline are counted in an array C, and

    B_start_index[I_B] = sum_{k < I_B} C[k]                                                 (Eq. 2)

gives where each baseline's run starts in the re-ordered data.  PAPER.md:73 says "according to eq. (2)" for
the baseline number; that is a typo for Eq. (1) (R14).  "Ordered by time" = input row order kept
within a baseline (rows arrive in time order), i.e. a STABLE re-order.

Plain numpy, written in the paper's order: index, count, prefix sum, stable placement.
"""
import numpy as np


def baseline_index(ant1, ant2, n_ant):
    """Eq. (1), element-wise, int64."""
    a1 = np.asarray(ant1, dtype=np.int64)
    a2 = np.asarray(ant2, dtype=np.int64)
    S = np.minimum(a1, a2)
    return (-S * S + 2 * S * n_ant + S) // 2 + np.abs(a1 - a2)


def n_baseline_slots(n_ant):
    """Number of values Eq. (1) can take: N_ant (N_ant + 1) / 2 (autocorrelation slots included)."""
    return n_ant * (n_ant + 1) // 2


def start_index(ant1, ant2, n_ant):
    """C (samples per baseline) and Eq. (2): (C, B_start_index), both of length n_baseline_slots + 1
    (last entry of B_start_index = number of rows)."""
    ib = baseline_index(ant1, ant2, n_ant)
    nb = n_baseline_slots(n_ant)
    C = np.zeros(nb, dtype=np.int64)
    for k in ib:                       # "count the number of timestamps under the same baseline number"
        C[k] += 1
    B = np.zeros(nb + 1, dtype=np.int64)
    for k in range(nb):                # Eq. (2)
        B[k + 1] = B[k] + C[k]
    return C, B


def reorder(ant1, ant2, n_ant):
    """perm with perm[slot] = input row: rows grouped by I_B, input (time) order kept inside a group."""
    ib = baseline_index(ant1, ant2, n_ant)
    _, B = start_index(ant1, ant2, n_ant)
    cursor = B[:-1].copy()
    perm = np.empty(ib.size, dtype=np.int64)
    for row, k in enumerate(ib):       # sequential placement: stable by construction
        perm[cursor[k]] = row
        cursor[k] += 1
    return perm
