"""GPU parity tests (-m gpu) of the relaxing-TVD step (gamer_rtvd_step) against the fp64 oracle
oracle/rtvd_oracle.hpp, element by element in the R14 metric, through the C ABI."""
import numpy as np
import pytest
import torch

import parity_util as pu
import paper_1007_3818_b200 as gh
from harness import metrics
from harness import workloads as wl
from oracle import rtvd_oracle as R

pytestmark = pytest.mark.gpu
G = wl.GAMMA
DEV = "cuda:0"
TOL1, TOL10 = 1e-4, 1e-3


def run_gpu(groups, dt, dx, sweep):
    x = torch.from_numpy(np.ascontiguousarray(groups)).to(DEV)
    out = torch.full((x.shape[0], 5, 16, 16, 16), float("nan"), dtype=torch.float32, device=DEV)
    gh.gamer_rtvd_step(x, out, None, 16, 3, dt, dx, G, sweep)
    torch.cuda.synchronize()
    return out.cpu().numpy()


@pytest.mark.parametrize("sweep", [0, 1])
def test_random_states_one_step(sweep):
    """Independent random positive states in every stored cell: every limiter branch, every ghost cell matters."""
    g = wl.random_groups(7, seed=201, ghost=3)
    dt, dx = pu.f32(1.5e-3), pu.f32(1 / 16)
    out = run_gpu(g, dt, dx, sweep)
    ref, _ = R.step_groups(g, 16, dt, dx, G, sweep)
    assert np.isfinite(out).all()
    assert metrics.max_rel_err(out, ref, G) <= TOL1


def test_uniform_moving_state_preserved_exactly():
    U = wl.prim_box_to_cons(*(np.full((1, 1, 1), x) for x in (1.3, 0.37, -0.61, 0.23, 0.9))).astype(np.float32).reshape(5)
    g = np.broadcast_to(U[None, :, None, None, None], (3, 5, 22, 22, 22)).copy()
    for sweep in (0, 1):
        assert np.array_equal(run_gpu(g, pu.f32(4e-3), pu.f32(1 / 32), sweep), g[:, :, 3:-3, 3:-3, 3:-3])


def test_many_groups_ragged_tail_and_determinism():
    n = 2 * 148 + 37
    g = wl.random_groups(n, seed=202, ghost=3)
    dt, dx = pu.f32(1.5e-3), pu.f32(1 / 16)
    out = run_gpu(g, dt, dx, 0)
    sample = np.r_[0:3, 147:150, 295:298, n - 3:n]
    ref, _ = R.step_groups(g[sample], 16, dt, dx, G, 0)
    assert metrics.max_rel_err(out[sample], ref, G) <= TOL1
    assert np.array_equal(run_gpu(g[150:151], dt, dx, 0)[0], out[150])      # independent of the batch
    assert np.array_equal(run_gpu(g, dt, dx, 0), out)


def test_cfg2_turbulence_ten_alternating_steps_and_conservation():
    """The smooth turbulent box of configs[2] (64^3 here), ten steps with alternating sweep order, host-driven: parity
    with the oracle on the same dt sequence (1e-3 after ten steps) and conservation in the periodic box."""
    w = wl.config_2_turbulence(64, seed=2)
    dx = pu.f32(w.dx)
    Ug, Uo = w.U.copy(), w.U.astype(np.float64)
    for s in range(10):
        dt = wl.cfl_dt(Ug, w.dx, 0.5)
        Ug = wl.assemble_box(run_gpu(wl.cut_groups(Ug, w.bc, ghost=3), dt, dx, s % 2), w.shape)
        o, _ = R.step_groups(wl.cut_groups(Uo, w.bc, ghost=3), 16, dt, dx, G, s % 2)
        Uo = wl.assemble_box(o, w.shape)
        if s == 0:
            assert metrics.max_rel_err(Ug[None], Uo[None], G) <= TOL1
    assert metrics.max_rel_err(Ug[None], Uo[None], G) <= TOL10
    for q in range(5):
        s0, s1 = w.U[q].astype(np.float64).sum(), Ug[q].astype(np.float64).sum()
        assert abs(s1 - s0) <= 1e-5 * np.abs(w.U[q]).astype(np.float64).sum()


def test_sod_tube_transverse_momentum_stays_zero():
    w = wl.config_1_sod_tube(nx=256)
    dx = pu.f32(w.dx)
    U = w.U.copy()
    for s in range(20):
        dt = wl.cfl_dt(U, w.dx, 0.5)
        U = wl.assemble_box(run_gpu(wl.cut_groups(U, w.bc, ghost=3), dt, dx, s % 2), w.shape)
    assert np.all(U[2] == 0) and np.all(U[3] == 0)
    assert U[0].max() <= 1.0 + 1e-6 and U[0].min() >= 0.125 - 1e-6


def test_argument_errors():
    x = torch.ones((1, 5, 22, 22, 22), device=DEV)
    out = torch.zeros((1, 5, 16, 16, 16), device=DEV)
    for kw in (dict(dt=0.0), dict(dx=-1.0), dict(gamma=1.0), dict(sweep=2)):
        args = dict(dt=1e-3, dx=1e-2, gamma=G, sweep=0)
        args.update(kw)
        with pytest.raises(gh.GamerHydroError):
            gh.gamer_rtvd_step(x, out, 1, 16, 3, **args)
    with pytest.raises(gh.GamerHydroError):      # only ghost = 3 is served
        gh.gamer_rtvd_step(torch.ones((1, 5, 24, 24, 24), device=DEV), out, 1, 16, 4, 1e-3, 1e-2, G, 0)
    gh.gamer_rtvd_step(torch.zeros((0, 5, 22, 22, 22), device=DEV), torch.zeros((0, 5, 16, 16, 16), device=DEV), 0, 16, 3,
                       1e-3, 1e-2, G, 0)           # empty batch is a no-op


def _nonpositive(U):
    """Cells with rho <= 0 or P <= 0 in a [..., 5, z, y, x]-like array (fp64 arithmetic)."""
    U = np.asarray(U, dtype=np.float64)
    rho, mx, my, mz, E = (np.take(U, q, axis=-4) for q in range(5))
    P = (G - 1.0) * (E - 0.5 * (mx * mx + my * my + mz * mz) / rho)
    return int(((rho <= 0) | (P <= 0)).sum())


def test_the_field_the_bench_times_all_4096_groups_both_sweep_orders_and_ten_steps():
    """bench.py's relaxing-TVD leg runs on the Mach-30 field of configs[3] at 256^3 cut
    with three ghost cells (4096 groups, 28 per persistent CTA) — this is that input (same recipe, seed, dt and dx as
    bench.py), ALL 4096 groups element by element against the fp64 oracle: one step in either sweep order within 1e-4,
    then ten steps with alternating order within 1e-3. fp32 pressure from E - ke at Mach 30 with the max(P, 0) clamp of
    RT6 is where a relaxing-TVD kernel could drift from its oracle. Output finite; non-positive cells are counted on
    both sides and must agree (RT6: no floors anywhere, so the count is part of the result)."""
    w = wl.config_3_cosmo(256, seed=3)
    dx = pu.f32(w.dx)
    grp = wl.cut_groups(w.U, w.bc, ghost=3)
    assert grp.shape == (4096, 5, 22, 22, 22)
    dt = pu.f32(w.dt())
    for sweep in (0, 1):
        out = run_gpu(grp, dt, dx, sweep)
        ref, _ = R.step_groups(grp, 16, dt, dx, G, sweep)
        assert np.isfinite(out).all()
        err = metrics.max_rel_err(out, ref, G)
        bad_gpu, bad_ref = _nonpositive(out), _nonpositive(ref)
        print("rtvd cfg3 256^3 sweep %d: max rel err %.3e, non-positive cells gpu %d / oracle %d" % (sweep, err, bad_gpu, bad_ref))
        assert err <= TOL1, (sweep, err)
        assert bad_gpu == bad_ref
    Ug, Uo = w.U.copy(), w.U.astype(np.float64)
    for s in range(10):
        dt = wl.cfl_dt(Ug, w.dx, 0.5)
        Ug = wl.assemble_box(run_gpu(wl.cut_groups(Ug, w.bc, ghost=3), dt, dx, s % 2), w.shape)
        o, _ = R.step_groups(wl.cut_groups(Uo, w.bc, ghost=3), 16, dt, dx, G, s % 2)
        Uo = wl.assemble_box(o, w.shape)
        assert np.isfinite(Ug).all(), s
    err10 = metrics.max_rel_err(Ug[None], Uo[None], G)
    print("rtvd cfg3 256^3 ten alternating steps: max rel err %.3e, non-positive cells gpu %d / oracle %d"
          % (err10, _nonpositive(Ug), _nonpositive(Uo)))
    assert err10 <= TOL10, err10
