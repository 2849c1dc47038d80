"""Pins for the oracle's index computation (oracle/ig_oracle.c: orc_index).

Expected values are worked by hand from PAPER.md eq 4.2 (:1081-1089:
-du/2 < delta_u <= du/2), the nearest-sample rule of eq 2.11-2.12 (:546-556, ties
toward -inf: DESIGN.md reading 2), the sqrt(w) plane spacing (:633, :1068) and the
conjugate rule eq 4.10 (:1416-1427). None of them re-types the oracle's formula.
"""
import numpy as np
import pytest

C = 299792458.0


def _exact_setup(orc, grid_n=256, beta=8):
    """Find a cell size for which the oracle's scale constant ku is exactly 2^-k, so
    that hand-chosen sample coordinates are reproduced with no rounding."""
    base = 1.0 / (grid_n * (beta / (C * 2.0 ** -24)))     # du = beta*2^24/c  ->  ku ~ 2^-24
    x = base
    for _ in range(2000):
        ku, _ = orc.constants(grid_n, x, beta, 1, 0.0)
        if ku == 2.0 ** -24:
            return x
        x = np.nextafter(x, np.inf if ku < 2.0 ** -24 else -np.inf)
    pytest.skip("no exact cell size found")


# fu (oversampled-sample units) -> (U nearest sample, cell x, offset) for beta = 8
HAND = [
    (0.0, 0, 0, 0), (0.49, 0, 0, 0), (0.5, 0, 0, 0), (0.51, 1, 0, 1), (-0.5, -1, 0, -1),
    (-0.49, 0, 0, 0), (3.4, 3, 0, 3), (3.5, 3, 0, 3), (3.6, 4, 0, 4), (4.5, 4, 0, 4),
    (4.6, 5, 1, -3), (-3.4, -3, 0, -3), (-3.5, -4, -1, 4), (-4.5, -5, -1, 3), (8.0, 8, 1, 0),
    (12.0, 12, 1, 4), (12.6, 13, 2, -3), (-11.5, -12, -2, 4), (-12.5, -13, -2, 3), (100.25, 100, 12, 4),
    (101.0, 101, 13, -3),
]


def test_hand_table_eq_4_2(orc):
    n, beta = 256, 8
    cell = _exact_setup(orc, n, beta)
    fu = np.array([h[0] for h in HAND])
    # u_m * nu = fu * 2^24 exactly (nu = 2^24 Hz, u_m = fu), times ku = 2^-24 -> fu exactly
    uvw = np.stack([fu, -fu, np.zeros_like(fu)], 1)
    idx = orc.index_records(uvw, [2.0 ** 24], n, cell, beta, 1, 0.0, [7])
    for i, (f, U, x, off) in enumerate(HAND):
        assert idx["X"][i, 0] == x + n // 2, (f, "X")
        assert idx["off_u"][i, 0] == off, (f, "off_u")
        assert x * beta + off == U
    # the v axis got -fu: its nearest sample is ceil(-fu - 1/2), worked here by integer logic
    for i, (f, _, _, _) in enumerate(HAND):
        twice = round(-2 * f * 100)            # exact in hundredths
        V = -((-(twice - 100)) // 200)         # ceil((twice-100)/200)
        y = (V + 3) // 8
        assert idx["Y"][i, 0] == y + n // 2 and idx["off_v"][i, 0] == V - 8 * y, f


@pytest.mark.parametrize("beta", [1, 2, 3, 4, 8])
def test_offset_range_and_identity(orc, beta):
    rng = np.random.default_rng(5)
    n = 512
    du = 30.0
    cell = 1.0 / (n * du)
    uvw = rng.uniform(-0.45 * n * du, 0.45 * n * du, (4000, 3))
    idx = orc.index_records(uvw, [C, 1.5 * C], n, cell, beta, 1, 0.0, [7])
    lo = -((beta - 1) // 2)                                     # offsets in (-beta/2, beta/2]
    assert idx["off_u"].min() >= lo and idx["off_u"].max() <= beta // 2
    assert set(np.unique(idx["off_u"])) == set(range(lo, beta // 2 + 1))
    # cell*beta + offset is the nearest oversampled sample of the true coordinate
    sgn = np.where(uvw[:, 2] < 0, -1.0, 1.0)
    for c, lam_inv in enumerate([1.0, 1.5]):
        true_u = sgn * uvw[:, 0] * lam_inv / du * beta
        U = (idx["X"][:, c] - n // 2) * beta + idx["off_u"][:, c]
        assert np.abs(U - true_u).max() <= 0.5 + 1e-9


def test_conjugate_flip_symmetry(orc):
    rng = np.random.default_rng(6)
    n, beta, P, wmax = 512, 8, 16, 900.0
    du = 25.0
    uvw = rng.uniform(-4000, 4000, (3000, 3))
    uvw[:, 2] = rng.uniform(-wmax, wmax, 3000)
    sup = 7 + 2 * np.arange(P)
    a = orc.index_records(uvw, [C], n, 1 / (n * du), beta, P, wmax, sup)
    b = orc.index_records(-uvw, [C], n, 1 / (n * du), beta, P, wmax, sup)
    for k in ("X", "Y", "off_u", "off_v", "plane"):
        assert np.array_equal(a[k], b[k]), k
    assert np.array_equal(a["flags"] & 1, (uvw[:, 2:3] < 0).astype(np.int32))
    assert np.all((a["flags"] & 1) ^ (b["flags"] & 1))      # w=0 never drawn here


def test_w_zero_is_not_flipped(orc):
    idx = orc.index_records([[100.0, -50.0, 0.0], [100.0, -50.0, -0.0]], [C], 256, 1 / (256 * 20.0), 8, 4, 100.0, [7, 9, 11, 13])
    assert np.all((idx["flags"] & 1) == 0) and np.all(idx["plane"] == 0)
    assert idx["X"][0, 0] == 128 + 5 and idx["Y"][0, 0] == 128 - 3   # 100/20 = 5 cells, -50/20 -> -2.5 -> cell -3? see below
    # -50 lambda = -2.5 cells = sample -20 of 8 -> cell floor((-20+3)/8) = -3, offset 4  (eq 4.2: delta <= du/2)
    assert idx["off_v"][0, 0] == 4 and idx["off_u"][0, 0] == 0


def test_plane_nearest_in_sqrt_w(orc):
    P, wmax = 33, 5000.0
    sup = np.full(P, 7)
    p = np.arange(P - 1)
    w_lo = wmax * ((p + 0.49) / (P - 1)) ** 2          # just below the midpoint in sqrt(w): plane p
    w_hi = wmax * ((p + 0.51) / (P - 1)) ** 2          # just above: plane p+1
    w_on = wmax * (np.arange(P) / (P - 1)) ** 2        # on the plane
    for w, want in ((w_lo, p), (w_hi, p + 1), (w_on, np.arange(P))):
        uvw = np.stack([np.zeros_like(w), np.zeros_like(w), w], 1)
        idx = orc.index_records(uvw, [C], 256, 1 / (256 * 20.0), 8, P, wmax, sup)
        assert np.array_equal(idx["plane"][:, 0], want)
        idx = orc.index_records(-uvw, [C], 256, 1 / (256 * 20.0), 8, P, wmax, sup)
        assert np.array_equal(idx["plane"][:, 0], want)
    idx = orc.index_records([[0, 0, 3 * wmax]], [C], 256, 1 / (256 * 20.0), 8, P, wmax, sup)
    assert idx["plane"][0, 0] == P - 1                 # clamped (reading 4)
    # frequency scales w in wavelengths: doubling nu at w_max/4 metres... plane of w=w_max/2 lambda
    idx = orc.index_records([[0, 0, wmax / 4]], [2 * C], 256, 1 / (256 * 20.0), 8, P, wmax, sup)
    assert idx["plane"][0, 0] == round(np.sqrt(0.5) * (P - 1))


def test_edge_records_dropped_whole(orc):
    n, beta, du = 64, 8, 10.0
    S = 7                                              # h = 3: centre cells 3..60 are on-grid
    xs = np.arange(-40, 40)
    uvw = np.stack([xs * du, np.zeros_like(xs, dtype=float), np.zeros_like(xs, dtype=float)], 1).astype(float)
    idx = orc.index_records(uvw, [C], n, 1 / (n * du), beta, 1, 0.0, [S])
    X = idx["X"][:, 0]
    on = (idx["flags"][:, 0] & 2) != 0
    assert np.array_equal(on, (X >= 3) & (X <= 60))


def test_non_finite_coordinates_are_dropped(orc):
    """DESIGN.md reading 20: a NaN or infinite u, v or w has no cell; the record is off the grid (bit1 clear) and its
    tuple is zero apart from the conj bit, for every channel; finite neighbours are unaffected (:1278 drop rule)."""
    n, beta, P = 64, 8, 4
    good = [1.0, 2.0, 3.0]
    uvw = np.array([good, [np.nan, 2, 3], [1, np.inf, -3], [1, 2, np.nan], [1, 2, -np.inf], good])
    idx = orc.index_records(uvw, [3e8, 2e8], n, 1e-3, beta, P, 100.0, [7, 7, 9, 9])
    for r in (1, 2, 3, 4):
        for k in ("X", "Y", "off_u", "off_v", "plane"):
            assert (idx[k][r] == 0).all(), (r, k)
        assert ((idx["flags"][r] & 2) == 0).all()
    assert idx["flags"][2, 0] == 1 and idx["flags"][4, 0] == 1 and idx["flags"][1, 0] == 0
    for k in idx:
        assert (idx[k][0] == idx[k][5]).all()
    assert (idx["flags"][0] & 2).all()
    # and the gridder leaves them out of grid, normaliser and the gridded count
    vis = np.ones((6, 2, 1), np.complex64); wt = np.ones((6, 2, 1), np.float32)
    bank = np.ones((49 + 49 + 81 + 81) * beta * beta, dtype=np.complex128)
    off = np.cumsum([0, 49, 49, 81]) * beta * beta
    g, nrm, st = orc.grid_records(idx, vis, wt, n, beta, [7, 7, 9, 9], bank, off)
    assert st[0] == 4 and st[1] == 8
