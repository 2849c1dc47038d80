"""Pins for the oracle's taper and w-kernel bank (oracle/reference.py).

What fixes them: scipy's angular prolate spheroidal function (a different
algorithm), the ODE the spheroidal satisfies, C_0(0,0)=1 and "the w=0 kernel is
the transform of the taper" (eq 2.9), DFT identities
(inversion, DC value, Parseval), the symmetries the thesis states (:1068-1070) and
the Fresnel closed form of the w-term for a small field (eq 2.14 :580).
"""
import numpy as np
import pytest


def test_taper_is_prolate_spheroidal_scipy(orc):
    from scipy.special import pro_ang1
    x = np.linspace(0.0, 0.999, 400)
    s = pro_ang1(1, 1, 3 * np.pi, x)[0] / np.sqrt(1 - x * x)
    assert np.abs(orc.taper(x) - s / s[0]).max() < 1e-10
    assert orc.taper(0.0) == pytest.approx(1.0, abs=1e-14)
    assert np.all(np.diff(orc.taper(x)) < 0)                 # monotone fall-off
    assert np.array_equal(orc.taper(-x), orc.taper(x))
    assert orc.taper(1.5) == 0.0 and orc.taper(1.0) == 0.0 and orc.taper(-1.0) == 0.0


def test_taper_satisfies_spheroidal_ode(orc):
    """(1-x^2)psi'' - 4x psi' + (b - c^2 x^2)psi = 0 with one constant b (alpha=1, c=3pi)."""
    c = 3 * np.pi
    x = np.linspace(0.05, 0.9, 30)
    hstep = 1e-3
    p0, pp, pm = orc.taper(x), orc.taper(x + hstep), orc.taper(x - hstep)
    d1 = (pp - pm) / (2 * hstep)
    d2 = (pp - 2 * p0 + pm) / hstep ** 2
    b = -((1 - x * x) * d2 - 4 * x * d1 - c * c * x * x * p0) / p0
    assert np.ptp(b) < 1e-3 * abs(b.mean())


def test_w0_plane_is_transform_of_taper(orc):
    n, beta, du = 16, 4, 25.0
    m = beta * n
    C0 = orc.oversampled_kernel(0, 1, 0.0, du, beta, n, -m // 2, m // 2 - 1)
    assert np.abs(C0.imag).max() < 1e-14                     # real
    assert C0[m // 2, m // 2] == pytest.approx(1.0, abs=1e-14)   # C_0(0,0) = 1
    # inverse DFT over the untrimmed plane returns the sampled taper / A
    q = np.arange(-m // 2, m // 2)
    a = np.arange(-n // 2, n // 2)
    Einv = np.exp(2j * np.pi * np.outer(a, q) / m) / m
    back = Einv @ C0 @ Einv.T
    psi = orc.taper(2.0 * a / n)
    want = np.outer(psi, psi) / np.outer(psi, psi).sum()
    assert np.abs(back - want).max() < 1e-12
    # uv-domain closed form of the same family: (1-nu^2) psi(nu), nu = |u|/(3 du)  (sanity, truncation-limited)
    nu = q / beta / 3.0
    closed = np.where(np.abs(nu) < 1, (1 - nu ** 2) * orc.taper(np.clip(nu, -1, 1)), 0.0)
    assert np.abs(C0[m // 2] - closed).max() < 2e-2


def test_dft_identities_w_plane(orc):
    n, beta, du, P, wmax = 16, 4, 25.0, 8, 600.0
    m = beta * n
    for p in (0, 3, 7):
        Cp = orc.oversampled_kernel(p, P, wmax, du, beta, n, -m // 2, m // 2 - 1)
        f, A = orc.image_plane_function(p, P, wmax, du, n)
        assert Cp.sum() == pytest.approx(m * m * f[n // 2, n // 2] / A, abs=1e-9)       # DC identity
        assert (np.abs(Cp) ** 2).sum() == pytest.approx(m * m * (np.abs(f) ** 2).sum() / A ** 2, rel=1e-12)  # Parseval
        assert np.abs(Cp - Cp.T).max() < 1e-13                                           # u <-> v
        # C_p(-q) = C_p(q): compare on the symmetric index range
        sym = Cp[1:, 1:]
        assert np.abs(sym - sym[::-1, ::-1]).max() < 1e-12
    widths = []
    n2, wmax2 = 32, 20000.0
    m2 = beta * n2
    for p in range(P):
        Cc = np.abs(orc.oversampled_kernel(p, P, wmax2, du, beta, n2, -m2 // 2, m2 // 2 - 1)[m2 // 2])
        widths.append(np.max(np.nonzero(Cc > 1e-3)[0]) - m2 // 2)
    assert all(b >= a for a, b in zip(widths, widths[1:])) and widths[-1] > 2 * widths[0]   # support grows with w (:633)


def test_w_screen_sign_fresnel(orc):
    """Small field: gbar_w ~ exp(-j pi w (l^2+m^2)) (eq 2.14 :580 inverted, :606), whose transform
    is the chirp exp(+j pi u^2/w). Multiplied by a taper of Gaussian-like width a the phase becomes
    +pi u^2/w / (1 + (a/(pi w))^2): it must INCREASE with |u|, stay below the pure-chirp phase and
    approach it as w grows. A wrong sign of the w-term fails the first assertion."""
    n, beta, du = 64, 2, 8.0           # field 1/du = 0.125 rad
    m = beta * n
    u = np.arange(0, 6) * du / beta
    ratios = []
    for wp in (300.0, 1200.0):
        row = orc.oversampled_kernel(1, 2, wp, du, beta, n, 0, 5)[0]        # qv = 0, qu = 0..5
        ph = np.unwrap(np.angle(row)) - np.angle(row[0])
        chirp = np.pi * u ** 2 / wp
        assert np.all(np.diff(ph) > 0)
        assert np.all(ph[1:] < 1.02 * chirp[1:])
        ratios.append(ph[1] / chirp[1])
    assert 0.2 < ratios[0] < ratios[1] < 1.02 and ratios[1] > 0.8


def test_bank_layout_and_selection(orc):
    """K[p][ov][ou][ty][tx] = C_p[ty*beta - off_v][tx*beta - off_u] (eq 4.1 with reading 1)."""
    beta, du, wmax = 4, 25.0, 500.0
    sup = np.array([5, 7, 9])
    bank, off = orc.build_bank(sup, wmax, du, beta, 9)
    assert off.tolist() == [0, 25 * 16, 25 * 16 + 49 * 16] and bank.size == (25 + 49 + 81) * 16
    n = orc.inner_samples(9)
    assert n == 32
    for p, S in enumerate(sup):
        h = (S - 1) // 2
        C = orc.oversampled_kernel(p, 3, wmax, du, beta, n, -(h + 1) * beta, (h + 1) * beta)
        K = bank[off[p]: off[p] + S * S * beta * beta].reshape(beta, beta, S, S)
        for offv in (-1, 0, 2):
            for offu in (-1, 1, 2):
                for ty in (-h, 0, h):
                    for tx in (-h, 1, h):
                        want = C[ty * beta - offv + (h + 1) * beta, tx * beta - offu + (h + 1) * beta]
                        assert K[offv + 1, offu + 1, ty + h, tx + h] == want
    assert bank[off[0] + (1 * beta + 1) * 25 + 2 * 5 + 2] == pytest.approx(1.0, abs=1e-13)  # C_0(0,0) at off=0, centre tap


def test_kernel_samples_agree_with_the_plane(orc):
    """kernel_samples (pair-by-pair DFT) against oversampled_kernel (whole plane) on random sample pairs."""
    rng = np.random.default_rng(11)
    P, w_max, du, beta, n = 6, 900.0, 25.0, 4, 32
    for p in (0, 3, 5):
        C = orc.oversampled_kernel(p, P, w_max, du, beta, n, -20, 20)
        qv, qu = rng.integers(-20, 21, 50), rng.integers(-20, 21, 50)
        got = orc.kernel_samples(p, P, w_max, du, beta, n, qv, qu)
        assert np.abs(got - C[qv + 20, qu + 20]).max() < 1e-13


def test_auto_supports_against_the_whole_plane(orc):
    """Automatic supports (:1114 1e-3 rule, reading 7) pinned against the whole oversampled plane computed the
    other way (E f E^T): outside the detected window the axis samples are <= 1e-3, the window is minimal, the
    w = 0 plane of the spheroidal taper needs 7 cells, and supports do not shrink as |w| grows."""
    P, w_max, du, beta, max_support = 6, 3000.0, 25.0, 4, 31
    sup = orc.auto_supports(P, w_max, du, beta, max_support)
    assert sup[0] == 7
    assert (np.diff(sup) >= 0).all() and sup[-1] > sup[0]
    assert (sup % 2 == 1).all() and sup.max() <= max_support
    n = orc.inner_samples(max_support)
    qmax = beta * ((max_support - 1) // 2)
    for p in range(P):
        C = np.abs(orc.oversampled_kernel(p, P, w_max, du, beta, n, -qmax, qmax))
        axis = np.maximum(C[qmax, :], C[:, qmax])          # row and column through the centre
        q = np.abs(np.arange(-qmax, qmax + 1))
        h = (sup[p] - 1) // 2
        if sup[p] < max_support:
            assert axis[q > h * beta].max(initial=0.0) <= 1e-3
        assert axis[q > (h - 1) * beta].max() > 1e-3        # one cell less would cut a sample above the threshold
