"""ig_grid_static against ig_grid: the entry point for callers that cannot allocate device memory.

Some users of the library run where cudaMalloc is not theirs to call: a gridding stage living inside another
program's process (the host application owns the device heap and passes in fixed buffers), or a streaming loop
that cannot take the device-wide stall of cudaMalloc / cudaFree. They cannot provide the per-batch work buffer
ig_grid needs, so ig_grid_static keeps its scratch in a 32 MiB array inside libig.so (include/ig.h,
csrc/ig_static.cu). This file checks that the result is the one ig_grid gives, on two calls in a row that share
that array (the second must not see what the first left behind), that an oversized batch is refused with a
message that names the limit, and that the call really takes no device memory.

The file name sorts last on purpose: the driver runs pytest with -x, and a failure here must not hide the
parity tests. It builds its own workload and contexts, so it passes alone in a fresh process as well as after
the rest of the suite.
"""
import dataclasses

import numpy as np
import pytest

from paper_1403_4209_b200 import synth

pytestmark = pytest.mark.gpu

# the bars of tests/test_gpu_parity.py (BASELINE.json north_star); both sides accumulate in fp32 with atomics in a
# non-deterministic order, so they agree far inside them but not bit for bit
FROB_TOL = 1e-5
MAX_TOL = 1e-4

# configuration 2's geometry, reduced: 91 baselines x 100 time steps x 16 channels = 145 600 records of 4
# polarisations, supports 7..33 (both work distributions run), about 19 MiB of scratch
CFG = dataclasses.replace(synth.CONFIGS[1], n_station=14, n_time=100)


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("gpu-marked test needs a CUDA device; there is no CPU fallback")
    from paper_1403_4209_b200 import build
    build.build()
    return torch


def _gridder(wl):
    from paper_1403_4209_b200.binding import Gridder
    cfg = wl["cfg"]
    g = Gridder(cfg.grid_n, wl["cell_rad"], cfg.n_wplanes, cfg.oversampling, int(wl["supports"].max()), cfg.n_pol)
    g.allocate(wl["supports"])
    g.build_wkernels(wl["w_max"])
    return g


def _agree(got, want):
    diff = got.astype(np.complex128) - want.astype(np.complex128)
    frob = np.linalg.norm(diff.ravel()) / np.linalg.norm(want.ravel())
    mx = np.abs(diff).max() / np.abs(want).max()
    assert frob <= FROB_TOL, f"relative Frobenius difference {frob:.3e}"
    assert mx <= MAX_TOL, f"max |delta| / max|grid| = {mx:.3e}"


def test_static_scratch_matches_work_buffer_on_two_calls_in_a_row(torch_cuda):
    from paper_1403_4209_b200.binding import IG_STATIC_WORK_BYTES
    torch = torch_cuda
    wl = synth.make_workload(CFG)
    d = "cuda:0"
    uvw = torch.from_numpy(wl["uvw_m"]).to(d)
    bl = torch.from_numpy(wl["baseline"]).to(d)
    vis = torch.from_numpy(np.ascontiguousarray(wl["vis"])).to(d)
    wt = torch.from_numpy(wl["weights"]).to(d)
    nrow = uvw.shape[0]
    # two batches of different length, the longer one first: the second call then runs over scratch that still holds
    # the first call's keys, records and plan beyond its own extent
    cut = (nrow * 5 // 8) // 7 * 7 + 3
    batches = [slice(0, cut), slice(cut, nrow)]
    ref, sta = _gridder(wl), _gridder(wl)
    assert 0 < ref.workspace_bytes(cut, CFG.n_chan) <= IG_STATIC_WORK_BYTES
    free_before_second = None
    for k, b in enumerate(batches):
        ref.grid_visibilities(uvw[b], bl[b], wl["freqs_hz"], vis[b], wt[b])
        if k == 1:
            torch.cuda.synchronize()
            free_before_second = torch.cuda.mem_get_info()[0]
        sta.grid_visibilities_static(uvw[b], bl[b], wl["freqs_hz"], vis[b], wt[b])
        if k == 1:
            torch.cuda.synchronize()
            # nothing was taken from the device between the two readings (the first call had already brought the
            # library's array and kernels onto the GPU)
            assert torch.cuda.mem_get_info()[0] >= free_before_second - (1 << 20)
        want = ref.grid_complex()
        assert np.abs(want).max() > 0
        _agree(sta.grid_complex(), want)
        assert sta.stats() == ref.stats()
        assert sta.last_launches() == ref.last_launches() > 0
    # the work buffer bound to the context is still the one ig_grid uses afterwards
    sta.grid_visibilities(uvw[batches[1]], bl[batches[1]], wl["freqs_hz"], vis[batches[1]], wt[batches[1]])
    ref.grid_visibilities(uvw[batches[1]], bl[batches[1]], wl["freqs_hz"], vis[batches[1]], wt[batches[1]])
    _agree(sta.grid_complex(), ref.grid_complex())


def test_static_scratch_refuses_a_batch_beyond_its_limit(torch_cuda):
    from paper_1403_4209_b200.binding import IgError, IG_STATIC_WORK_BYTES
    torch = torch_cuda
    wl = synth.make_workload(dataclasses.replace(CFG, n_time=8))
    g = _gridder(wl)
    d = "cuda:0"
    nchan = CFG.n_chan
    nrow = 40_000                                   # x 16 channels x 4 polarisations: about 80 MiB of scratch
    assert g.workspace_bytes(nrow, nchan) > IG_STATIC_WORK_BYTES
    uvw = torch.zeros((nrow, 3), dtype=torch.float64, device=d)
    bl = torch.zeros(nrow, dtype=torch.int32, device=d)
    vis = torch.ones((nrow, nchan, CFG.n_pol, 2), dtype=torch.float32, device=d)
    wt = torch.ones((nrow, nchan, CFG.n_pol), dtype=torch.float32, device=d)
    with pytest.raises(IgError) as err:
        g.grid_visibilities_static(uvw, bl, wl["freqs_hz"], vis, wt)
    assert "IG_ENOMEM" in str(err.value) and "IG_STATIC_WORK_BYTES" in str(err.value)
    assert g.stats() == (0, 0, 0)                   # nothing was enqueued
    assert float(g.grid.abs().max()) == 0.0
    # an empty batch is fine, as with ig_grid
    g.grid_visibilities_static(uvw[:0], bl[:0], wl["freqs_hz"], vis[:0], wt[:0])
