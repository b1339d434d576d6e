"""Shared helpers of the GPU parity tests: run the oracle and the CUDA path on the same seeded float32
inputs and compare element by element with the R14 metric (harness/metrics.py), with the guard-disagreement
accounting of reading R7."""
import numpy as np
import torch

from harness import metrics
import paper_1007_3818_b200 as gh
from oracle import mhm_oracle as O

NEAR_GUARD = metrics.NEAR_GUARD
MAX_EXCLUDED_FRACTION = 1e-5
suspect_mask = metrics.suspect_mask


def f32(x):
    return float(np.float32(x))


def run_gpu(groups, dt, dx, gamma, limiter, path=gh.PATH_AUTO, want_bflux=True, N=16, ghost=2, guard_map=None):
    """groups: numpy [G,5,S,S,S] float32 or float64 -> (U_out, bflux, (guard, nonpos)) as numpy. guard_map: a list
    that receives the kernel's map of the cells that fell back to first order, uint8 [G,N+2,N+2,N+2]."""
    dev = torch.device("cuda", 0)
    x = torch.from_numpy(np.ascontiguousarray(groups)).to(dev)
    G = x.shape[0]
    out = torch.full((G, 5, N, N, N), float("nan"), dtype=x.dtype, device=dev)
    bf = torch.full((G, 6, 5, N, N), float("nan"), dtype=x.dtype, device=dev) if want_bflux else None
    gh.gamer_hydro_status()
    gh.gamer_hydro_set_path(path)
    gm = torch.zeros((G, N + 2, N + 2, N + 2), dtype=torch.uint8, device=dev) if guard_map is not None else None
    if gm is not None:
        gh.gamer_hydro_set_guard_map(gm)
    try:
        fn = gh.gamer_hydro_step if x.dtype == torch.float32 else gh.gamer_hydro_step_f64
        fn(x, out, bf, G, N, ghost, dt, dx, gamma, limiter)
        torch.cuda.synchronize()
    finally:
        gh.gamer_hydro_set_path(gh.PATH_AUTO)
        if gm is not None:
            gh.gamer_hydro_set_guard_map(None)
            guard_map.append(gm.cpu().numpy())
    st = gh.gamer_hydro_status()
    return out.cpu().numpy(), (bf.cpu().numpy() if want_bflux else None), st


def disagreement_mask(gpu_guard, oracle_guard):
    """Interior cells whose update can be touched by a guard DISAGREEMENT (reading R7): the cells where exactly one of
    GPU and oracle fell back to first order, and their six face neighbours. Both maps: uint8 [G,N+2,N+2,N+2]."""
    d = (gpu_guard != 0) != (oracle_guard != 0)
    m = d.copy()
    m[:, 1:] |= d[:, :-1]; m[:, :-1] |= d[:, 1:]
    m[:, :, 1:] |= d[:, :, :-1]; m[:, :, :-1] |= d[:, :, 1:]
    m[:, :, :, 1:] |= d[:, :, :, :-1]; m[:, :, :, :-1] |= d[:, :, :, 1:]
    return m[:, 1:-1, 1:-1, 1:-1]


def compare(groups, dt, dx, gamma, limiter, gpu_out, gpu_bf=None, N=16, ghost=2, gpu_guard=None):
    """Oracle on the same inputs -> dict(err, err_bflux, excluded_fraction, oracle=StepResult). With the kernel's
    guard map the excluded cells are those where GPU and oracle actually disagree on the guard (R7); without it, the
    conservative superset of cells whose oracle margin is within NEAR_GUARD of zero."""
    r = O.step_groups(groups, N, ghost, dt, dx, gamma, limiter)
    sus = disagreement_mask(gpu_guard, r.guard) if gpu_guard is not None else suspect_mask(r.margin, N)
    keep = ~sus[:, None]
    err = metrics.max_rel_err(gpu_out, r.U_out, gamma, mask=np.broadcast_to(keep, r.U_out.shape))
    res = dict(err=err, excluded_fraction=float(sus.mean()), oracle=r, suspect=sus)
    if gpu_bf is not None:
        e = metrics.bflux_errors(gpu_bf, r.bflux, r.U_out, gamma)
        face_sus = [sus[:, :, :, 0], sus[:, :, :, -1], sus[:, :, 0, :], sus[:, :, -1, :], sus[:, 0], sus[:, -1]]
        for f in range(6):
            e[:, f] = np.where(face_sus[f][:, None], 0.0, e[:, f])
        res["err_bflux"] = float(e.max())
    return res
