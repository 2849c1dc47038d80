"""Thin ctypes binding over the C-ABI library libig.so (include/ig.h).

Argument marshalling only: every step of the path runs in the library's CUDA kernels.
PyTorch owns device memory and the stream. There is no CPU fallback: `load()` raises if
the library has not been built, and compute calls raise IgError on any failure.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB = None

IG_STATIC_WORK_BYTES = 32 << 20    # include/ig.h: scratch built into the library for ig_grid_static
STATUS = {0: "IG_OK", 1: "IG_EINVAL", 2: "IG_ESTATE", 3: "IG_ECUDA", 4: "IG_ENOMEM", 5: "IG_EUNSUPPORTED"}

_vp, _sz, _ll, _i, _d = C.c_void_p, C.c_size_t, C.c_longlong, C.c_int, C.c_double
# name -> (restype, argtypes); mirrors include/ig.h one to one
SIGNATURES = {
    "ig_create": (_i, [C.POINTER(_vp), _i, _d, _i, _i, _i, _i]),
    "ig_destroy": (None, [_vp]),
    "ig_last_error": (C.c_char_p, [_vp]),
    "ig_grid_bytes": (_sz, [_vp]),
    "ig_workspace_bytes": (_sz, [_vp, _ll, _i]),
    "ig_bank_bytes": (_sz, [_vp, _vp]),
    "ig_finalize_workspace_bytes": (_sz, [_vp]),
    "ig_bind": (_i, [_vp, _vp, _sz, _vp, _sz, _vp, _sz, _vp]),
    "ig_build_wkernels": (_i, [_vp, _d, _vp]),
    "ig_get_supports": (_i, [_vp, _vp]),
    "ig_debug_set_wkernels": (_i, [_vp, _d, _vp, _vp, _sz]),
    "ig_debug_get_wkernels": (_i, [_vp, _vp, _sz]),
    "ig_grid": (_i, [_vp, _vp, _vp, _ll, _vp, _i, _vp, _vp]),
    "ig_grid_static": (_i, [_vp, _vp, _vp, _ll, _vp, _i, _vp, _vp]),
    "ig_host_staging_bytes": (_sz, [_vp, _ll, _i]),
    "ig_set_host_slices": (_i, [_vp, _i]),
    "ig_grid_host": (_i, [_vp, _vp, _vp, _ll, _vp, _i, _vp, _vp]),
    "ig_finalize": (_i, [_vp, _vp, _vp]),
    "ig_set_per_channel_grids": (_i, [_vp, _i]),
    "ig_finalize_channel": (_i, [_vp, _i, _vp, _vp]),
    "ig_get_stats": (_i, [_vp, C.POINTER(_ll), C.POINTER(_ll), C.POINTER(_ll)]),
    "ig_get_commits": (_i, [_vp, C.POINTER(_ll)]),
    "ig_set_compression": (_i, [_vp, _i]),
    "ig_get_compressed": (_i, [_vp, C.POINTER(_ll)]),
    "ig_set_commit_counting": (_i, [_vp, _i]),
    "ig_measure_fp32_peak": (_i, [_vp, _vp, C.POINTER(_d)]),
    "ig_set_sort_tile_shift": (_i, [_vp, _i]),
    "ig_set_gather_min_support": (_i, [_vp, _i]),
    "ig_set_stokes_output": (_i, [_vp, _i]),
    "ig_measure_commit_rate": (_i, [_vp, _vp, _sz, _i, C.POINTER(_d)]),
    "ig_get_timing": (_i, [_vp, _i, C.POINTER(C.c_float), C.POINTER(C.c_float)]),
    "ig_get_gridder_split": (_i, [_vp, _i, C.POINTER(C.c_float), C.POINTER(C.c_float)]),
    "ig_reset_accumulators": (_i, [_vp]),
    "ig_last_launches": (_i, [_vp]),
    "ig_debug_indices": (_i, [_vp, _vp, _ll, _vp, _i, _vp, _vp, _vp, _vp, _vp, _vp]),
    "ig_debug_taper": (_i, [_vp, _i, _vp]),
}


class IgError(RuntimeError):
    pass


def lib_path() -> str:
    return os.path.join(_HERE, "libig.so")


def load():
    """Load libig.so. Fails loudly if it is missing (run `python -m paper_1403_4209_b200.build`)."""
    global _LIB
    if _LIB is None:
        path = lib_path()
        if not os.path.exists(path):
            raise IgError(f"{path} not built: run __graft_entry__.build() or python paper_1403_4209_b200/build.py; "
                          "there is no CPU fallback")
        lib = C.CDLL(path)
        for name, (res, args) in SIGNATURES.items():
            fn = getattr(lib, name)
            fn.restype, fn.argtypes = res, args
        _LIB = lib
    return _LIB


def _np_ptr(a: np.ndarray):
    return a.ctypes.data_as(_vp)


def taper(eta) -> np.ndarray:
    """psi(eta) as the library computes it (host code, no GPU needed)."""
    eta = np.ascontiguousarray(eta, dtype=np.float64)
    out = np.empty_like(eta)
    st = load().ig_debug_taper(_np_ptr(eta), eta.size, _np_ptr(out))
    if st:
        raise IgError(STATUS.get(st, str(st)))
    return out


class Gridder:
    """One context = one grid. Device buffers are torch tensors owned by this object."""

    def __init__(self, grid_n, cell_rad, n_wplanes, oversampling, max_support, n_pol, device="cuda:0",
                 stream=None):
        import torch
        self.torch = torch
        self.lib = load()
        self.device = torch.device(device)
        self.grid_n, self.n_pol, self.n_wplanes, self.beta = grid_n, n_pol, n_wplanes, oversampling
        self.max_support = max_support
        self.ctx = _vp()
        st = self.lib.ig_create(C.byref(self.ctx), grid_n, cell_rad, n_wplanes, oversampling, max_support, n_pol)
        if st:
            raise IgError(f"ig_create: {STATUS.get(st, st)}")
        self.stream = stream
        self.grid = None
        self.work = None
        self.bank = None
        self.supports = None

    # -- plumbing ---------------------------------------------------------------------
    def _check(self, st, what):
        if st:
            msg = self.lib.ig_last_error(self.ctx)
            raise IgError(f"{what}: {STATUS.get(st, st)}: {msg.decode() if msg else ''}")

    def _stream_ptr(self):
        s = self.stream if self.stream is not None else self.torch.cuda.current_stream(self.device)
        return _vp(s.cuda_stream)

    def _bind(self):
        self._check(self.lib.ig_bind(self.ctx, _vp(self.grid.data_ptr()), self.grid.numel() * 4,
                                     _vp(self.work.data_ptr()), self.work.numel(),
                                     _vp(self.bank.data_ptr()), self.bank.numel(), self._stream_ptr()), "ig_bind")

    def allocate(self, supports, work_bytes=0, n_channel_grids=0):
        """Allocate grid (zeroed), bank and a work buffer of at least `work_bytes`.
        n_channel_grids > 0: one grid per channel (ig_set_per_channel_grids)."""
        t = self.torch
        if supports is not None:
            supports = np.ascontiguousarray(supports, dtype=np.int32)
            assert supports.size == self.n_wplanes
        self.supports = supports          # None: automatic supports, known after build_wkernels
        with t.cuda.device(self.device):
            shape = (self.grid_n, self.grid_n, self.n_pol, 2)
            self.n_channel_grids = int(n_channel_grids)
            if self.n_channel_grids > 0:
                shape = (self.n_channel_grids,) + shape
            self.grid = t.zeros(shape, dtype=t.float32, device=self.device)
            nb = self.lib.ig_bank_bytes(self.ctx, _np_ptr(supports) if supports is not None else None)
            self.bank = t.empty(nb, dtype=t.uint8, device=self.device)
            need = max(int(work_bytes), self.lib.ig_workspace_bytes(self.ctx, 0, 1), 1 << 20)
            self.work = t.empty(need, dtype=t.uint8, device=self.device)
        self._bind()
        if self.n_channel_grids > 0:
            self._check(self.lib.ig_set_per_channel_grids(self.ctx, 1), "ig_set_per_channel_grids")

    def finalize_channel(self, channel):
        t = self.torch
        self.ensure_work(self.lib.ig_finalize_workspace_bytes(self.ctx))
        img = t.empty((self.n_pol, self.grid_n, self.grid_n), dtype=t.float32, device=self.device)
        norm = np.zeros(self.n_pol, dtype=np.float64)
        self._check(self.lib.ig_finalize_channel(self.ctx, int(channel), _vp(img.data_ptr()), _np_ptr(norm)), "ig_finalize_channel")
        return img, norm

    def channel_grid_complex(self, channel) -> np.ndarray:
        """Grid of one channel as complex64 numpy [N][N][npol] (per-channel grid mode)."""
        self.torch.cuda.synchronize(self.device)
        g, n = self.grid[channel], self.grid_n
        if self.n_pol == 4:
            g = g.reshape(2, n, n, 2, 2).permute(1, 2, 0, 3, 4).reshape(n, n, 4, 2)
        return g.contiguous().cpu().numpy().view(np.complex64)[..., 0]

    def ensure_work(self, nbytes):
        if self.work is None or self.work.numel() < nbytes:
            self.work = None
            self.work = self.torch.empty(int(nbytes), dtype=self.torch.uint8, device=self.device)
            self._bind()

    def workspace_bytes(self, nrow, nchan, host=False):
        n = self.lib.ig_workspace_bytes(self.ctx, nrow, nchan)
        if host:
            n += self.lib.ig_host_staging_bytes(self.ctx, nrow, nchan)
        return n

    # -- the calls of include/ig.h ----------------------------------------------------
    def build_wkernels(self, w_max):
        tab = _np_ptr(self.supports) if self.supports is not None else None
        self._check(self.lib.ig_build_wkernels(self.ctx, float(w_max), tab), "ig_build_wkernels")
        out = np.zeros(self.n_wplanes, dtype=np.int32)
        self._check(self.lib.ig_get_supports(self.ctx, _np_ptr(out)), "ig_get_supports")
        self.supports = out

    def debug_set_wkernels(self, w_max, bank_c64: np.ndarray):
        b = np.ascontiguousarray(bank_c64, dtype=np.complex64)
        self._check(self.lib.ig_debug_set_wkernels(self.ctx, float(w_max), _np_ptr(self.supports), _np_ptr(b),
                                                   b.nbytes), "ig_debug_set_wkernels")

    def debug_get_wkernels(self) -> np.ndarray:
        n = int((self.supports.astype(np.int64) ** 2).sum()) * self.beta * self.beta
        out = np.empty(n, dtype=np.complex64)
        self._check(self.lib.ig_debug_get_wkernels(self.ctx, _np_ptr(out), out.nbytes), "ig_debug_get_wkernels")
        return out

    def _check_inputs(self, uvw_m, baseline_id, vis, weights, nrow, nchan, on_device):
        """The C ABI takes bare pointers: dtype, density, element count and residence are checked here."""
        t = self.torch
        want = (("uvw_m", uvw_m, ("float64",), nrow * 3), ("baseline_id", baseline_id, ("int32",), nrow),
                ("vis", vis, ("float32", "complex64"), None), ("weights", weights, ("float32",), nrow * nchan * self.n_pol))
        for name, a, dtypes, numel in want:
            is_t = isinstance(a, t.Tensor)
            dt = str(a.dtype).replace("torch.", "")
            if dt not in dtypes:
                raise IgError(f"{name}: dtype {dt}, expected {dtypes}")
            if numel is None:
                numel = nrow * nchan * self.n_pol * (1 if dt == "complex64" else 2)
            n = a.numel() if is_t else a.size
            if n != numel:
                raise IgError(f"{name}: {n} elements, expected {numel}")
            if not (a.is_contiguous() if is_t else a.flags["C_CONTIGUOUS"]):
                raise IgError(f"{name}: not contiguous")
            if on_device and not (is_t and a.is_cuda and a.device == self.device):
                raise IgError(f"{name}: must be a tensor on {self.device}")
            if not on_device and is_t and a.is_cuda:
                raise IgError(f"{name}: must be host memory")

    def grid_visibilities(self, uvw_m, baseline_id, freqs_hz, vis, weights):
        """Device tensors: uvw_m f64 [nrow,3], baseline_id i32 [nrow], vis c64/f32 [nrow,nchan,npol(,2)],
        weights f32 [nrow,nchan,npol]; freqs_hz: host numpy f64."""
        freqs = np.ascontiguousarray(freqs_hz, dtype=np.float64)
        nrow, nchan = int(uvw_m.shape[0]), int(freqs.size)
        self._check_inputs(uvw_m, baseline_id, vis, weights, nrow, nchan, on_device=True)
        self.ensure_work(self.workspace_bytes(nrow, nchan))
        self._check(self.lib.ig_grid(self.ctx, _vp(uvw_m.data_ptr()), _vp(baseline_id.data_ptr()), nrow,
                                     _np_ptr(freqs), nchan, _vp(vis.data_ptr()), _vp(weights.data_ptr())), "ig_grid")

    def grid_visibilities_static(self, uvw_m, baseline_id, freqs_hz, vis, weights):
        """ig_grid_static: same arguments and result as grid_visibilities, but the scratch is the library's built-in
        32 MiB device array instead of a work buffer, so nothing is allocated here or in the library. For callers
        that may not touch the device heap (see include/ig.h). Raises IgError (IG_ENOMEM) when the batch is too large."""
        freqs = np.ascontiguousarray(freqs_hz, dtype=np.float64)
        nrow, nchan = int(uvw_m.shape[0]), int(freqs.size)
        self._check_inputs(uvw_m, baseline_id, vis, weights, nrow, nchan, on_device=True)
        self._check(self.lib.ig_grid_static(self.ctx, _vp(uvw_m.data_ptr()), _vp(baseline_id.data_ptr()), nrow,
                                            _np_ptr(freqs), nchan, _vp(vis.data_ptr()), _vp(weights.data_ptr())), "ig_grid_static")

    def grid_visibilities_host(self, uvw_m, baseline_id, freqs_hz, vis, weights):
        """Same with HOST buffers (numpy arrays or pinned CPU torch tensors): the end-to-end call."""
        freqs = np.ascontiguousarray(freqs_hz, dtype=np.float64)
        nrow, nchan = int(uvw_m.shape[0]), int(freqs.size)
        self._check_inputs(uvw_m, baseline_id, vis, weights, nrow, nchan, on_device=False)
        self.ensure_work(self.workspace_bytes(nrow, nchan, host=True))
        ptr = lambda a: _vp(a.data_ptr()) if hasattr(a, "data_ptr") else _np_ptr(a)
        self._check(self.lib.ig_grid_host(self.ctx, ptr(uvw_m), ptr(baseline_id), nrow, _np_ptr(freqs), nchan,
                                          ptr(vis), ptr(weights)), "ig_grid_host")

    def finalize(self):
        t = self.torch
        self.ensure_work(self.lib.ig_finalize_workspace_bytes(self.ctx))
        img = t.empty((self.n_pol, self.grid_n, self.grid_n), dtype=t.float32, device=self.device)
        norm = np.zeros(self.n_pol, dtype=np.float64)
        self._check(self.lib.ig_finalize(self.ctx, _vp(img.data_ptr()), _np_ptr(norm)), "ig_finalize")
        return img, norm

    def stats(self):
        g, d, u = _ll(), _ll(), _ll()
        self._check(self.lib.ig_get_stats(self.ctx, C.byref(g), C.byref(d), C.byref(u)), "ig_get_stats")
        return g.value, d.value, u.value

    def set_host_slices(self, n: int):
        self._check(self.lib.ig_set_host_slices(self.ctx, int(n)), "ig_set_host_slices")

    def set_gather_min_support(self, s: int):
        self._check(self.lib.ig_set_gather_min_support(self.ctx, int(s)), "ig_set_gather_min_support")

    def set_stokes_output(self, on: bool):
        self._check(self.lib.ig_set_stokes_output(self.ctx, int(bool(on))), "ig_set_stokes_output")

    def set_sort_tile_shift(self, shift: int):
        self._check(self.lib.ig_set_sort_tile_shift(self.ctx, int(shift)), "ig_set_sort_tile_shift")

    def set_compression(self, on: bool):
        self._check(self.lib.ig_set_compression(self.ctx, int(bool(on))), "ig_set_compression")

    def compressed(self) -> int:
        n = _ll()
        self._check(self.lib.ig_get_compressed(self.ctx, C.byref(n)), "ig_get_compressed")
        return n.value

    def set_commit_counting(self, on: bool):
        self._check(self.lib.ig_set_commit_counting(self.ctx, int(bool(on))), "ig_set_commit_counting")

    def commits(self) -> int:
        n = _ll()
        self._check(self.lib.ig_get_commits(self.ctx, C.byref(n)), "ig_get_commits")
        return n.value

    def measure_fp32_peak(self) -> float:
        v = _d()
        sink = self.torch.zeros(1, dtype=self.torch.float32, device=self.device)
        self._check(self.lib.ig_measure_fp32_peak(self._stream_ptr(), _vp(sink.data_ptr()), C.byref(v)), "ig_measure_fp32_peak")
        return v.value

    def measure_commit_rate(self, nbytes, run_len=8) -> float:
        """1e9 pixel commits/s into a scratch buffer of nbytes (see include/ig.h)."""
        buf = self.torch.zeros(int(nbytes) // 4, dtype=self.torch.float32, device=self.device)
        v = _d()
        self._check(self.lib.ig_measure_commit_rate(self._stream_ptr(), _vp(buf.data_ptr()), buf.numel() * 4, run_len,
                                                    C.byref(v)), "ig_measure_commit_rate")
        return v.value

    def timing(self, calls_back=0):
        """(ingest_ms, gridder_ms) of the ig_grid call `calls_back` calls ago."""
        a, b = C.c_float(), C.c_float()
        self._check(self.lib.ig_get_timing(self.ctx, calls_back, C.byref(a), C.byref(b)), "ig_get_timing")
        return a.value, b.value

    def gridder_split(self, calls_back=0):
        """(moving-window ms, gather-phase ms) of the gridder time of that ig_grid call."""
        a, b = C.c_float(), C.c_float()
        self._check(self.lib.ig_get_gridder_split(self.ctx, calls_back, C.byref(a), C.byref(b)), "ig_get_gridder_split")
        return a.value, b.value

    def reset(self):
        self.grid.zero_()
        self._check(self.lib.ig_reset_accumulators(self.ctx), "ig_reset_accumulators")

    def last_launches(self) -> int:
        return int(self.lib.ig_last_launches(self.ctx))

    def debug_indices(self, uvw_m, freqs_hz):
        t = self.torch
        freqs = np.ascontiguousarray(freqs_hz, dtype=np.float64)
        nrow, nchan = int(uvw_m.shape[0]), int(freqs.size)
        outs = [t.empty((nrow, nchan), dtype=t.int32, device=self.device) for _ in range(6)]
        self._check(self.lib.ig_debug_indices(self.ctx, _vp(uvw_m.data_ptr()), nrow, _np_ptr(freqs), nchan,
                                              *[_vp(o.data_ptr()) for o in outs]), "ig_debug_indices")
        return dict(zip(("X", "Y", "off_u", "off_v", "plane", "flags"), [o.cpu().numpy() for o in outs]))

    def grid_complex(self) -> np.ndarray:
        """The grid as complex64 numpy [N][N][npol] (synchronises); undoes the 4-pol pair-plane layout."""
        self.torch.cuda.synchronize(self.device)
        g = self.grid
        if self.n_pol == 4:
            n = self.grid_n
            g = g.view(2, n, n, 2, 2).permute(1, 2, 0, 3, 4).reshape(n, n, 4, 2)
        return g.contiguous().cpu().numpy().view(np.complex64)[..., 0]

    def grid_window_complex(self, x0, y0, w, h) -> np.ndarray:
        """Pixels [y0, y0+h) x [x0, x0+w) of the grid as complex64 numpy [h][w][npol] (synchronises)."""
        self.torch.cuda.synchronize(self.device)
        n = self.grid_n
        if self.n_pol == 4:
            g = self.grid.view(2, n, n, 2, 2)[:, y0:y0 + h, x0:x0 + w].permute(1, 2, 0, 3, 4).reshape(h, w, 4, 2)
        else:
            g = self.grid[y0:y0 + h, x0:x0 + w]
        return g.contiguous().cpu().numpy().view(np.complex64)[..., 0]

    def touched_pixels(self) -> int:
        """Pixels with a non-zero value in any polarisation (synchronises)."""
        t, n = self.torch, self.grid_n
        grids = self.grid if getattr(self, "n_channel_grids", 0) > 0 else [self.grid]     # per-channel mode: summed over the grids
        total = 0
        for one in grids:
            g = one.reshape(2, n * n, 4) if self.n_pol == 4 else one.reshape(1, n * n, self.n_pol * 2)
            hit = t.zeros(n * n, dtype=t.bool, device=self.device)
            for part in g:
                for lo in range(0, n * n, 1 << 26):
                    hit[lo:lo + (1 << 26)] |= (part[lo:lo + (1 << 26)] != 0).any(dim=1)
            total += int(hit.sum().item())
        return total

    def close(self):
        if self.ctx:
            self.lib.ig_destroy(self.ctx)
            self.ctx = _vp()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
