"""Pins of oracle/track_commits.py, the oracle-side commit model behind bench.py's roofline.

The model's closed form (pixels leaving an S x S window that moves by (dx, dy)) is checked against a literal simulation
of Romein's ownership (Fig 2.1: a thread owns the grid points congruent to its residues modulo S and
commits its sum when its point leaves the window), and the stored numbers against a fresh run of the script's own
function on the two configurations that finish in seconds."""
import numpy as np

from oracle import track_commits as tc
from paper_1403_4209_b200 import synth


def _simulate(X, Y, S, on):
    """One track, records in time order: the set of pixels the S*S threads hold; a pixel leaving the set is one commit."""
    held, held_s, commits = set(), 0, 0
    for x, y, s, ok in zip(X, Y, S, on):
        if not ok:
            commits += len(held); held, held_s = set(), 0
            continue
        h = (s - 1) // 2
        new = {(yy, xx) for yy in range(y - h, y + h + 1) for xx in range(x - h, x + h + 1)}
        if s != held_s:                       # support change: every residue is re-mapped, all sums commit (:1349)
            commits += len(held)
        else:
            commits += len(held - new)
        held, held_s = new, s
    return commits + len(held)                # end of the track


def test_closed_form_equals_literal_ownership_simulation():
    rng = np.random.default_rng(7)
    n_time, n_bl, nchan = 40, 3, 2
    X = np.cumsum(rng.integers(-3, 4, (n_time, n_bl, nchan)), axis=0) + 100
    Y = np.cumsum(rng.integers(-12, 13, (n_time, n_bl, nchan)), axis=0) + 100
    S = rng.choice([7, 7, 7, 9, 11], (n_time, n_bl, nchan))
    on = rng.random((n_time, n_bl, nchan)) > 0.05
    total, by_class, upd = tc.track_commits(X.reshape(-1, nchan), Y.reshape(-1, nchan), S.reshape(-1, nchan),
                                            on.reshape(-1, nchan), n_time, n_bl)
    want = sum(_simulate(X[:, b, c], Y[:, b, c], S[:, b, c], on[:, b, c]) for b in range(n_bl) for c in range(nchan))
    assert total == want
    assert by_class.sum() == total and upd.sum() == int((np.where(on, S, 0).astype(np.int64) ** 2).sum())


def test_stored_numbers_are_the_scripts_own():
    stored = {(e["config"], e["support_law"]): e for e in tc.load()["entries"]}
    assert len(stored) == 10 and {k[0] for k in stored} == {c.name for c in synth.CONFIGS}
    for i in (0, 1):
        fresh = tc.model_config(i, "w")
        assert fresh == stored[(fresh["config"], "w")]
    for e in stored.values():                 # a commit is charged at most once per held pixel
        assert 0 < e["pixel_commits"] <= e["pixel_updates"]
