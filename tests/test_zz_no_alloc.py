"""gamer_hydro_max_speed_noalloc: the signal-speed maximum for callers that must not cause a device allocation.

Who needs it. An AMR code that has handed all of the GPU's memory to its own patch pools cannot let this library
cudaMalloc behind its back (the call may fail hours into a run), and a time loop that overlaps copies and kernels on
several streams cannot take the device-wide stall that cudaMalloc / cudaFree bring. The ordinary entry point,
gamer_hydro_max_speed, allocates the library's status block on first use; the variant under test keeps its partial
maxima in a fixed 256.25 KiB array that is part of the library image (at most 65536 patch groups per call) and writes
the result to a device float the caller owns.

This file is named so that pytest collects it last: `pytest -x` stops at the first failure, and a failure here must
not hide the parity tests. The GPU test runs the new entry point BEFORE anything else touches the library, so it passes
alone in a fresh process (no gamer_hydro_alloc has run) as well as after the other test files (library long set up).
"""
import ctypes

import numpy as np
import pytest
import torch

import paper_1007_3818_b200 as gh
from harness import workloads as wl

DEV = "cuda:0"


def test_noalloc_limit_and_argument_checks_need_no_device():
    """The size limit and the pointer checks are answered before any CUDA call (so also on a box without a GPU)."""
    L = gh.binding.lib()
    limit = gh.gamer_hydro_max_speed_noalloc_limit()
    assert limit == 65536
    fake = ctypes.c_void_p(256)                                    # never dereferenced: the calls below are refused
    assert L.gamer_hydro_max_speed_noalloc(fake, limit + 1, 16, 2, 5 / 3, fake, None) == 5      # TOO_LARGE
    assert "65536" in gh.gamer_hydro_strerror(5) and "noalloc" in gh.gamer_hydro_strerror(5)
    assert L.gamer_hydro_max_speed_noalloc(None, 4, 16, 2, 5 / 3, fake, None) == 1              # null input
    assert L.gamer_hydro_max_speed_noalloc(fake, 4, 16, 2, 5 / 3, None, None) == 1              # null output
    assert L.gamer_hydro_max_speed_noalloc(fake, 0, 16, 2, 5 / 3, fake, None) == 1              # empty batch
    assert L.gamer_hydro_max_speed_noalloc(fake, 4, 16, 2, 1.0, fake, None) == 1                # gamma <= 1
    assert L.gamer_hydro_max_speed_noalloc(fake, 4, 16, 2, 5 / 3, ctypes.c_void_p(258), None) == 1   # misaligned


@pytest.mark.gpu
def test_noalloc_max_speed_matches_the_allocating_path_on_consecutive_calls():
    """Two calls in a row (and then more) on different fields and different batch sizes, each compared with
    gamer_hydro_max_speed and with the fp64 formula of the harness at the tolerances of
    test_gpu_multistep.py::test_max_speed_matches_the_fp64_formula. The second batch is SMALLER than the first, so
    a result built from what the first call left in the shared array (stale per-group maxima, a counter that was not
    cleared) would be wrong."""
    w_big = wl.config_2_turbulence(64, seed=4)                     # 64 groups, maximum ~ 17
    g_big = w_big.groups()
    g_small = np.ascontiguousarray(wl.config_3_cosmo(64, seed=9).groups()[:24])   # 24 groups, cold gas: maximum ~ 0.16
    fields = [(g_big, torch.from_numpy(g_big).to(DEV), 2e-6),
              (g_small, torch.from_numpy(g_small).to(DEV), 1e-4)]  # Mach-30 cells: P from a cancelling difference in fp32
    inter = torch.from_numpy(np.ascontiguousarray(g_small[:, :, 2:-2, 2:-2, 2:-2])).to(DEV)
    outs = [torch.full((1,), float("nan"), dtype=torch.float32, device=DEV) for _ in range(6)]
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())                  # stream and event exist before memory is measured
    torch.cuda.synchronize()

    # the new entry point first, back to back on one stream, before the allocating path has been used at all
    gh.gamer_hydro_max_speed_noalloc(fields[0][1], outs[0])
    gh.gamer_hydro_max_speed_noalloc(fields[1][1], outs[1])
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    gh.gamer_hydro_max_speed_noalloc(fields[0][1], outs[2])                       # big again after small
    gh.gamer_hydro_max_speed_noalloc(inter, outs[3], ghost=0)                     # a U_out array (no ghost shell)
    side.wait_stream(torch.cuda.current_stream())                                 # ordered after the calls above
    with torch.cuda.stream(side):
        gh.gamer_hydro_max_speed_noalloc(fields[1][1], outs[4], stream=side)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free_before, "the calls changed the amount of free device memory"
    got = [float(o.item()) for o in outs[:5]]

    for (grp, d_U, tol), idx in ((fields[0], (0, 2)), (fields[1], (1, 4))):
        ref64 = wl.max_signal_speed(grp[:, :, 2:-2, 2:-2, 2:-2])
        existing = gh.gamer_hydro_max_speed(d_U)
        for q in idx:
            assert np.isfinite(got[q]) and got[q] > 0.0
            assert abs(got[q] - existing) <= tol * existing, (q, got[q], existing)
            assert abs(got[q] - ref64) <= tol * ref64, (q, got[q], ref64)
        assert got[idx[0]] == got[idx[1]]                                         # same input, same bits
    assert got[0] > 10.0 * got[1]                                                 # the stale-maximum trap is real
    assert abs(got[3] - gh.gamer_hydro_max_speed(inter, ghost=0)) <= 1e-4 * got[3]
    assert got[3] == got[1]                                                       # ghost cells never enter the maximum

    # a NaN cell makes the maximum NaN (the rule the CFL check of gamer_hydro_advance relies on), and the next call on
    # clean data is clean again
    bad = fields[1][1].clone()
    bad[3, 0, 9, 9, 9] = float("nan")
    gh.gamer_hydro_max_speed_noalloc(bad, outs[5])
    gh.gamer_hydro_max_speed_noalloc(fields[1][1], outs[4])
    torch.cuda.synchronize()
    assert np.isnan(outs[5].item()) and float(outs[4].item()) == got[1]

    # beyond the fixed array: refused with its own error code, nothing enqueued, the output untouched
    too_many = gh.gamer_hydro_max_speed_noalloc_limit() + 1
    outs[5].fill_(-1.0)
    rc = gh.binding.lib().gamer_hydro_max_speed_noalloc(fields[1][1].data_ptr(), too_many, 16, 2, 5 / 3,
                                                        outs[5].data_ptr(), None)
    torch.cuda.synchronize()
    assert rc == 5 and outs[5].item() == -1.0
