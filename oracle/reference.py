"""ORACLE - test infrastructure only (see oracle/ig_oracle.c header).

Plain fp64 numpy statement of the parts of the path that are not the record
loop: taper, w-kernel bank, finaliser, brute-force direct-Fourier imager; plus
the ctypes wrapper over oracle/ig_oracle.c (index computation and gridding).
Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / reference
legs may import this. It imports nothing from paper_1403_4209_b200.

Citations are PAPER.md line : section / equation; "reading k" = DESIGN.md table.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB = None


def build(force: bool = False) -> str:
    """Compile oracle/ig_oracle.c with gcc (no FMA contraction, OpenMP)."""
    src = os.path.join(_HERE, "ig_oracle.c")
    so = os.path.join(_HERE, "libig_oracle.so")
    if force or not os.path.exists(so) or os.path.getmtime(so) < os.path.getmtime(src):
        subprocess.check_call(["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC",
                               src, "-o", so, "-lm"])
    return so


def _lib():
    global _LIB
    if _LIB is None:
        _LIB = ctypes.CDLL(build())
    return _LIB


def _p(a, t):
    return a.ctypes.data_as(ctypes.POINTER(t))


# ----------------------------------------------------------------------------
# Taper: the prolate-spheroidal gridding function family of Schwab that the
# thesis takes from casacore ("casagridsf"). Its coefficients are
# not in the paper (reading 6), so psi is computed from its defining property:
# psi_{alpha,0}(c, .) is the eigenfunction with the LARGEST eigenvalue of the
# finite weighted Fourier transform
#     mu * psi(eta) = int_{-1}^{1} (1-t^2)^alpha * exp(j*c*eta*t) * psi(t) dt
# (the most concentrated function: the uv kernel (1-nu^2)^alpha psi(nu) of width
# m cells has image-plane transform proportional to psi itself), alpha = 1,
# m = 6, c = pi*m/2 = 3*pi. Solved by Nystrom discretisation on Gauss-Legendre
# nodes; psi is even so only the cosine part survives. Normalised psi(0) = 1.
# ----------------------------------------------------------------------------
_TAPER_CACHE = {}


def _taper_nodes(c: float, alpha: int, nq: int = 96):
    key = (c, alpha, nq)
    if key not in _TAPER_CACHE:
        t, wq = np.polynomial.legendre.leggauss(nq)
        kern = np.cos(c * np.outer(t, t)) * (wq * (1.0 - t * t) ** alpha)[None, :]
        ev, vec = np.linalg.eig(kern)
        k = int(np.argmax(ev.real))
        _TAPER_CACHE[key] = (t, wq, vec[:, k].real.copy(), float(ev[k].real))
    return _TAPER_CACHE[key]


def taper(eta, c: float = 3.0 * np.pi, alpha: int = 1):
    """psi(eta) for |eta| < 1 (Nystrom extension of the eigenvector); 0 at and beyond the
    field edge |eta| >= 1 (reading 5: keeps the sampled image-plane function symmetric,
    hence the w=0 kernel real and C(-q) = C(q), :1068-1070)."""
    eta = np.asarray(eta, dtype=np.float64)
    t, wq, vec, mu = _taper_nodes(c, alpha)

    def ext(x):
        return (np.cos(c * np.multiply.outer(x, t)) * (wq * (1.0 - t * t) ** alpha * vec)).sum(-1) / mu

    out = ext(eta) / ext(np.zeros(()))
    return np.where(np.abs(eta) < 1.0, out, 0.0)


# ----------------------------------------------------------------------------
# W-kernel bank, Algorithm 4.1 as a direct DFT (no FFT):
#   f_p[b][a] = psi(eta_a) psi(eta_b) exp(+j 2 pi w_p (sqrt(1-l_a^2-m_b^2) - 1))
#               (taper x conjugate w-screen, eq 2.14 :580, eq 2.21 :606-615)
#   C_p[qv][qu] = (1/A) sum_{a,b} f_p[b][a] exp(-j 2 pi (qu a + qv b)/(beta n))
#   A = sum psi psi  =>  C_0[0][0] = 1 (:1114).
# n image-plane samples span the field of view 1/du (reading 5); zero padding by
# beta gives uv samples du/beta apart (:1066). w_p = w_max (p/(P-1))^2 (:633,:1068).
# ----------------------------------------------------------------------------
def inner_samples(max_support: int) -> int:
    n = 1
    while n < 2 * max_support:
        n *= 2
    return n


def wplane_w(p: int, n_wplanes: int, w_max: float) -> float:
    return 0.0 if n_wplanes == 1 else w_max * (p / (n_wplanes - 1)) ** 2


def image_plane_function(p, n_wplanes, w_max, du, n):
    a = np.arange(-n // 2, n // 2, dtype=np.float64)
    psi = taper(2.0 * a / n)
    lm = a / (n * du)
    r2 = lm[None, :] ** 2 + lm[:, None] ** 2
    nm1 = np.sqrt(np.maximum(0.0, 1.0 - r2)) - 1.0
    w = wplane_w(p, n_wplanes, w_max)
    f = np.outer(psi, psi) * np.exp(2j * np.pi * w * nm1)
    return f, float(np.outer(psi, psi).sum())


def oversampled_kernel(p, n_wplanes, w_max, du, beta, n, q_lo, q_hi):
    """C_p[qv][qu] for qu,qv in [q_lo, q_hi] (oversampled sample indices)."""
    f, A = image_plane_function(p, n_wplanes, w_max, du, n)
    a = np.arange(-n // 2, n // 2, dtype=np.float64)
    q = np.arange(q_lo, q_hi + 1, dtype=np.float64)
    E = np.exp(-2j * np.pi * np.outer(q, a) / (beta * n))   # [q][a]
    return (E @ f @ E.T) / A                                # [qv][qu]


def kernel_samples(p, n_wplanes, w_max, du, beta, n, qv, qu):
    """C_p at the listed oversampled sample pairs (qv[k], qu[k]) only: the same direct DFT as
    oversampled_kernel, evaluated pair by pair (used to check single grid pixels of full-size runs)."""
    f, A = image_plane_function(p, n_wplanes, w_max, du, n)
    a = np.arange(-n // 2, n // 2, dtype=np.float64)
    qv = np.asarray(qv, dtype=np.float64)
    qu = np.asarray(qu, dtype=np.float64)
    out = np.empty(qv.size, dtype=np.complex128)
    for s0 in range(0, qv.size, 256):               # bounded temporaries
        Ev = np.exp(-2j * np.pi * np.outer(qv[s0:s0 + 256], a) / (beta * n))   # [k][b]
        Eu = np.exp(-2j * np.pi * np.outer(qu[s0:s0 + 256], a) / (beta * n))   # [k][a]
        out[s0:s0 + 256] = np.einsum("kb,kb->k", Ev @ f, Eu) / A
    return out


def auto_supports(n_wplanes, w_max, du, beta, max_support, threshold=1e-3):
    """Automatic support per plane (reading 7): r = largest |q| on the u-axis row or the
    v-axis column through the centre with |C_p| > threshold (C_0(0,0) = 1), searched over
    |q| <= beta*(max_support-1)/2; S = 2*ceil(r/beta)+1."""
    n = inner_samples(int(max_support))
    qmax = beta * ((max_support - 1) // 2)
    q = np.arange(-qmax, qmax + 1)
    zero = np.zeros_like(q)
    out = np.empty(n_wplanes, dtype=np.int32)
    for p in range(n_wplanes):
        cu = np.abs(kernel_samples(p, n_wplanes, w_max, du, beta, n, zero, q))
        cv = np.abs(kernel_samples(p, n_wplanes, w_max, du, beta, n, q, zero))
        over = (cu > threshold) | (cv > threshold)
        r = int(np.abs(q[over]).max()) if over.any() else 0
        out[p] = min(max_support, 2 * (-(-r // beta)) + 1)
    return out


def build_bank(supports, w_max, du, beta, max_support, planes=None):
    """Returns (bank complex128 flat, bank_off int64[P]).
    K[p][ov][ou][ty][tx] = C_p[ty*beta - off_v][tx*beta - off_u], ty,tx in [-h,h],
    ov = off_v + ceil(beta/2) - 1 (eq 4.1 :1078 with reading 1; layout :1100-1108).
    planes: optional subset of plane indices to compute; the other planes of the bank stay zero
    (for checks of a window of a large grid that only a few planes reach)."""
    supports = np.asarray(supports, dtype=np.int64)
    P = supports.size
    n = inner_samples(int(max_support))
    shift = (beta + 1) // 2 - 1
    off = np.zeros(P, dtype=np.int64)
    off[1:] = np.cumsum(supports[:-1] ** 2 * beta * beta)
    bank = np.zeros(int((supports ** 2).sum() * beta * beta), dtype=np.complex128)
    for p in (range(P) if planes is None else sorted(set(int(x) for x in planes))):
        S = int(supports[p]); h = (S - 1) // 2
        qmax = h * beta + beta          # covers every ty*beta - off
        C = oversampled_kernel(p, P, w_max, du, beta, n, -qmax, qmax)
        t = np.arange(-h, h + 1) * beta
        blk = np.empty((beta, beta, S, S), dtype=np.complex128)
        for ov in range(beta):
            for ou in range(beta):
                qv = t - (ov - shift) + qmax
                qu = t - (ou - shift) + qmax
                blk[ov, ou] = C[np.ix_(qv, qu)]
        bank[off[p]:off[p] + blk.size] = blk.ravel()
    return bank, off


# ----------------------------------------------------------------------------
# Record loop (oracle/ig_oracle.c)
# ----------------------------------------------------------------------------
def constants(grid_n, cell_rad, beta, n_wplanes, w_max):
    ku, kw = ctypes.c_double(), ctypes.c_double()
    _lib().orc_constants(ctypes.c_int(grid_n), ctypes.c_double(cell_rad), ctypes.c_int(beta),
                         ctypes.c_int(n_wplanes), ctypes.c_double(w_max),
                         ctypes.byref(ku), ctypes.byref(kw))
    return ku.value, kw.value


def index_records(uvw_m, freqs_hz, grid_n, cell_rad, beta, n_wplanes, w_max, supports):
    """dict of int32 arrays [nrow][nchan]: X, Y, off_u, off_v, plane, flags."""
    uvw_m = np.ascontiguousarray(uvw_m, dtype=np.float64)
    freqs_hz = np.ascontiguousarray(freqs_hz, dtype=np.float64)
    supports = np.ascontiguousarray(supports, dtype=np.int32)
    nrow, nchan = uvw_m.shape[0], freqs_hz.size
    out = {k: np.empty((nrow, nchan), dtype=np.int32)
           for k in ("X", "Y", "off_u", "off_v", "plane", "flags")}
    i32 = ctypes.c_int32
    _lib().orc_index(ctypes.c_int64(nrow), ctypes.c_int(nchan), _p(uvw_m, ctypes.c_double),
                     _p(freqs_hz, ctypes.c_double), ctypes.c_int(grid_n), ctypes.c_double(cell_rad),
                     ctypes.c_int(beta), ctypes.c_int(n_wplanes), ctypes.c_double(w_max),
                     _p(supports, i32), _p(out["X"], i32), _p(out["Y"], i32), _p(out["off_u"], i32),
                     _p(out["off_v"], i32), _p(out["plane"], i32), _p(out["flags"], i32))
    return out


def grid_records(idx, vis, weights, grid_n, beta, supports, bank, bank_off, grid=None,
                 norm=None, stats=None):
    """Adds the records to `grid` (complex128 [N][N][npol]); returns (grid, norm, stats)."""
    vis = np.ascontiguousarray(vis, dtype=np.complex64)
    weights = np.ascontiguousarray(weights, dtype=np.float32)
    nrow, nchan, npol = vis.shape
    supports = np.ascontiguousarray(supports, dtype=np.int32)
    bank = np.ascontiguousarray(bank, dtype=np.complex128)
    bank_off = np.ascontiguousarray(bank_off, dtype=np.int64)
    if grid is None:
        grid = np.zeros((grid_n, grid_n, npol), dtype=np.complex128)
    if norm is None:
        norm = np.zeros(npol, dtype=np.float64)
    if stats is None:
        stats = np.zeros(3, dtype=np.int64)
    i32 = ctypes.c_int32
    ix = {k: np.ascontiguousarray(v, dtype=np.int32) for k, v in idx.items()}
    _lib().orc_grid(ctypes.c_int64(nrow), ctypes.c_int(nchan), ctypes.c_int(npol),
                    _p(vis, ctypes.c_float), _p(weights, ctypes.c_float),
                    _p(ix["X"], i32), _p(ix["Y"], i32), _p(ix["off_u"], i32), _p(ix["off_v"], i32),
                    _p(ix["plane"], i32), _p(ix["flags"], i32), ctypes.c_int(grid_n),
                    ctypes.c_int(beta), _p(supports, i32), _p(bank_off, ctypes.c_int64),
                    _p(bank, ctypes.c_double), _p(grid, ctypes.c_double),
                    _p(norm, ctypes.c_double), _p(stats, ctypes.c_int64))
    return grid, norm, stats


def threads() -> int:
    return int(_lib().orc_threads())


def set_threads(n: int) -> None:
    """Thread count of the following grid_records calls (timing the single-thread rate)."""
    _lib().orc_set_threads(ctypes.c_int(int(n)))


# ----------------------------------------------------------------------------
# Finaliser, Algorithm 4.6: inverse transform of the grid
# with the uv origin at pixel (N/2,N/2) (eq 2.8 :516, unnormalised, +j), divide by
# the normaliser (eq 4.5), by the taper (eq 2.9 :523, reading 14) and by the sinc
# of the nearest-sample lookup (eq 2.13 :561-564). numpy's FFT is the library primitive;
# shifts put the origin where the paper does. Step 2's Stokes conversion (:1660, :1668) is
# finalize_stokes below (the paper prints no formulas: reading 21).
# ----------------------------------------------------------------------------
def transform_grid(grid):
    """img[pol][b][a] = sum_{Y,X} grid[Y][X][pol] e^{+j2pi((X-N/2)a+(Y-N/2)b)/N}, a,b in [-N/2,N/2)."""
    g = np.moveaxis(np.asarray(grid, dtype=np.complex128), -1, 0)
    n = g.shape[-1]
    img = np.fft.ifft2(np.fft.ifftshift(g, axes=(-2, -1)), axes=(-2, -1)) * (n * n)
    return np.fft.fftshift(img, axes=(-2, -1))


def finalize(grid, norm, beta):
    n = grid.shape[0]
    a = np.arange(-n // 2, n // 2, dtype=np.float64)
    psi = taper(2.0 * a / n)
    snc = np.sinc(a / (n * beta))                  # np.sinc(x) = sin(pi x)/(pi x)
    corr = np.outer(psi * snc, psi * snc)
    img = transform_grid(grid).real
    with np.errstate(divide="ignore", invalid="ignore"):
        out = img / (np.asarray(norm)[:, None, None] * corr[None])
    out[:, corr == 0.0] = 0.0
    return out


# Step 2 of Algorithm 4.6, "Convert to multiple-Stokes image and normalise".
# The paper gives no formulas (reading 21): polarisations are taken as the linear-feed correlations
# of a LOFAR MeasurementSet in its order (XX, XY, YX, YY), whose relation to the Stokes visibilities is
# the textbook one, XX = I + Q, XY = U + jV, YX = U - jV, YY = I - Q; inverted per image pixel on the
# NORMALISED complex images D_p = img_p / N_p ("convert ... and normalise"):
#   4 pol: I = (D_XX + D_YY)/2, Q = (D_XX - D_YY)/2, U = (D_XY + D_YX)/2, V = (D_XY - D_YX)/(2j)
#   2 pol (XX, YY): I, Q as above;   1 pol: I = D_0 (the only Stokes "that can be calculated", :1660).
# The real part is taken after the combination (V needs the imaginary parts), then steps 3-4 as finalize.
# A polarisation whose normaliser is zero was flagged throughout (eq 4.5 sums weights x kernel sums, :1286), its
# grid is identically zero, and 0/0 has no value: it enters the combinations as D_p = 0 (reading 21).
def finalize_stokes(grid, norm, beta):
    n, npol = grid.shape[0], grid.shape[2]
    a = np.arange(-n // 2, n // 2, dtype=np.float64)
    psi = taper(2.0 * a / n)
    snc = np.sinc(a / (n * beta))
    corr = np.outer(psi * snc, psi * snc)
    nrm = np.asarray(norm, dtype=np.float64)
    d = transform_grid(grid)
    for p in range(npol):
        d[p] = d[p] / nrm[p] if nrm[p] != 0.0 else 0.0
    if npol == 4:
        st = np.stack([(d[0] + d[3]) / 2, (d[0] - d[3]) / 2, (d[1] + d[2]) / 2, (d[1] - d[2]) / 2j])
    elif npol == 2:
        st = np.stack([(d[0] + d[1]) / 2, (d[0] - d[1]) / 2])
    else:
        st = d
    with np.errstate(divide="ignore", invalid="ignore"):
        out = st.real / corr[None]
    out[:, corr == 0.0] = 0.0
    return out


# ----------------------------------------------------------------------------
# Brute-force direct-Fourier dirty image (adjoint of the measurement equation
# eq 1.14), tiny inputs only:
#   D[b][a] = Re sum_i wt_i V_i exp(+j 2 pi (u_i l_a + v_i m_b + w_i (n_ab - 1))) / sum_i wt_i
# ----------------------------------------------------------------------------
def direct_image(u, v, w, vis, wt, grid_n, du):
    a = np.arange(-grid_n // 2, grid_n // 2, dtype=np.float64)
    lm = a / (grid_n * du)
    l, m = lm[None, :], lm[:, None]
    nm1 = np.sqrt(np.maximum(0.0, 1.0 - l * l - m * m)) - 1.0
    img = np.zeros((grid_n, grid_n), dtype=np.float64)
    for ui, vi, wi, Vi, ei in zip(u, v, w, vis, wt):
        img += (ei * Vi * np.exp(2j * np.pi * (ui * l + vi * m + wi * nm1))).real
    return img / np.sum(wt)
