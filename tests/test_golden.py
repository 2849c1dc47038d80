"""Values the thesis prints, kept as text fixtures under tests/golden/ (each file cites its passage)."""
import os

import numpy as np

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def _rows(name):
    with open(os.path.join(GOLDEN, name)) as f:
        return [ln.split() for ln in f if ln.strip() and not ln.startswith("#")]


def test_update_counts_printed_in_the_thesis(orc):
    """eq 4.17c through the oracle: one record with an S x S kernel and npol polarisations."""
    for S, npol, want, *_ in _rows("update_counts.txt"):
        S, npol, want = int(S), int(npol), int(want)
        n = 1 << int(np.ceil(np.log2(S + 8)))
        sup = np.array([S], dtype=np.int32)
        bank = np.ones(S * S, dtype=np.complex128)                      # beta = 1: one matrix
        idx = dict(X=[[n // 2]], Y=[[n // 2]], off_u=[[0]], off_v=[[0]], plane=[[0]], flags=[[2]])
        vis = np.ones((1, 1, npol), dtype=np.complex64)
        wt = np.ones((1, 1, npol), dtype=np.float32)
        grid, norm, stats = orc.grid_records(idx, vis, wt, n, 1, sup, bank, np.zeros(1, dtype=np.int64))
        assert tuple(stats) == (1, 0, want)
        assert np.count_nonzero(grid) == want                           # each update lands on its own grid point


def test_fig_2_1_thread_layout():
    """Romein's distribution as the figure prints it: the thread of grid point (Y, X) is fixed by (Y mod S, X mod S).
    The CUDA gridder uses exactly this residue rule (lane owns the pixels congruent to its (i, j) modulo S), and the
    record header's (c, d) = (-a mod S, -b mod S) of eq 4.7 turns a tap of a footprint at (a, b) into that residue."""
    fig = np.array(_rows("fig2_1_threads.txt"), dtype=int)
    S = 3
    Y, X = np.mgrid[0:fig.shape[0], 0:fig.shape[1]]
    assert np.array_equal(fig, (Y % S) * S + (X % S) + 1)
    # footprint with top-left corner (b, a): tap (ty, tx) is served by the lane with residues ((b+ty) mod S, (a+tx) mod S);
    # with c = -a mod S the lane with residue i serves tap tx = (i + c) mod S - one lane per tap, all taps covered
    for a in range(0, 6):
        c = (-a) % S
        taps = sorted(((i + c) % S) for i in range(S))
        assert taps == list(range(S))
        for i in range(S):
            tx = (i + c) % S
            assert (a + tx) % S == i
