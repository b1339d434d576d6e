"""GPU parity tests (-m gpu) of BASELINE.json:configs[1], [2] and [4] AT THEIR STATED SIZES and step counts, run
device-resident through gamer_hydro_advance (fp32) or the fp64 step + ghost refill + signal-speed calls, against the
fp64 oracle stepped with the same time-step sequence, the exact Riemann solution (configs[1]) and the Sedov-Taylor
closed form (configs[4]). The scaled-down versions in test_gpu_parity.py are the fast ones; these take minutes."""
import os

import numpy as np
import pytest
import torch

import exact_riemann as er
import parity_util as pu
import paper_1007_3818_b200 as gh
from harness import metrics
from harness import workloads as wl
from oracle import mhm_oracle as O

pytestmark = pytest.mark.gpu
G = wl.GAMMA
DEV = "cuda:0"
BC = {"periodic": gh.BC_PERIODIC, "outflow": gh.BC_OUTFLOW}


def _grid(shape):
    nz, ny, nx = shape
    return (nx // 16, ny // 16, nz // 16)


def _golden(name):
    out = {}
    with open(os.path.join(os.path.dirname(__file__), "golden", name)) as f:
        for line in f:
            if line.strip() and not line.startswith("#"):
                k, v = line.split()[:2]
                out[k] = float(v)
    return out


class DeviceRun:
    """A uniform grid kept on the device. fp32: gamer_hydro_advance; fp64: signal speed -> dt (R15, not rounded) ->
    gamer_hydro_step_f64 -> gamer_hydro_fill_ghosts, all on device arrays."""

    def __init__(self, w, dtype):
        self.w, self.dtype = w, dtype
        self.grid, self.bc = _grid(w.shape), [BC[b] for b in w.bc]
        self.dx = pu.f32(w.dx) if dtype == np.float32 else w.dx
        self.d_U = torch.from_numpy(w.groups(dtype)).to(DEV)
        n = self.d_U.shape[0]
        self.d_out = torch.empty((n, 5, 16, 16, 16), dtype=self.d_U.dtype, device=DEV)
        self.dts = []

    def advance(self, steps):
        w = self.w
        if self.dtype == np.float32:
            self.dts += gh.gamer_hydro_advance(self.d_U, self.d_out, None, self.grid, steps, w.cfl, self.dx, bc=self.bc,
                                               gamma=G, limiter=w.limiter)
        else:
            for _ in range(steps):
                vmax = gh.gamer_hydro_max_speed(self.d_U, gamma=G)
                dt = w.cfl * self.dx / vmax
                gh.gamer_hydro_step_f64(self.d_U, self.d_out, None, None, 16, 2, dt, self.dx, G, w.limiter)
                gh.gamer_hydro_fill_ghosts(self.d_out, self.d_U, self.grid, bc=self.bc)
                self.dts.append(dt)
        torch.cuda.synchronize()

    def box(self):
        return wl.assemble_box(self.d_out.cpu().numpy(), self.w.shape)


def _oracle_advance(Uo, w, dts, dx):
    for dt in dts:
        r = O.step_groups(wl.cut_groups(Uo, w.bc), 16, 2, dt, dx, G, w.limiter, want_bflux=False, want_guard=False)
        Uo = wl.assemble_box(r.U_out, w.shape)
    return Uo


@pytest.mark.parametrize("limiter", [0, 1])
@pytest.mark.parametrize("dtype", [np.float32, np.float64])
def test_cfg1_sod_tube_1024_cells_64_groups_200_steps(dtype, limiter):
    """configs[1] as stated: 1024 x 16 x 16, 64 groups, 200 steps at C = 0.5, outflow along the tube. Oracle parity at
    steps 1, 10 and 200 (same dt sequence), L1(rho) against the exact Riemann solution at t = sum(dt), the star-state
    plateaus of SURVEY.md App. A, transverse momentum exactly zero."""
    w = wl.config_1_sod_tube(nx=1024, limiter=limiter, steps=200)
    run = DeviceRun(w, dtype)
    Uo = w.U.astype(np.float64)
    done = 0
    # north_star: 1e-4 after one step, 1e-3 after ten (fp32); 1e-11 (fp64). The 200-step mark is held to the same
    # bounds (measured on B200: 9.5e-7 in fp32, 1.2e-14 in fp64)
    tol = {np.float32: {1: 1e-4, 10: 1e-3, 200: 1e-3}, np.float64: {1: 1e-11, 10: 1e-11, 200: 1e-11}}[dtype]
    for mark in (1, 10, 200):
        run.advance(mark - done)
        Uo = _oracle_advance(Uo, w, run.dts[done:mark], run.dx)
        done = mark
        Ug = run.box()
        err = metrics.max_rel_err(Ug[None], Uo[None], G)
        print("cfg1 %s limiter %d step %d: max rel err %.3e" % (np.dtype(dtype).name, limiter, mark, err))
        assert err <= tol[mark], (mark, err)
        assert np.all(Ug[2] == 0) and np.all(Ug[3] == 0)         # transverse momentum stays exactly zero
    assert len(run.dts) == 200
    t = float(np.sum(np.asarray(run.dts, dtype=np.float64)))
    assert abs(t - 0.0187) < 0.002                                  # t about 0.0187 with R15
    # against the exact solution
    gold = _golden("sod_exact_gamma53.txt")
    nx = 1024
    x = (np.arange(nx) + 0.5) / nx
    xi = (x - 0.5) / t
    rho_e, u_e, p_e = er.sample(G, (1, 0, 1), (0.125, 0, 0.1), xi)
    U = Ug.astype(np.float64)
    assert np.array_equal(Ug[:, 3, 5, :], Ug[:, 11, 2, :])          # stays one-dimensional, bit for bit
    rho = U[0, 3, 5, :]
    l1 = float(np.mean(np.abs(rho - rho_e)))
    l1_oracle = float(np.mean(np.abs(Uo[0, 3, 5, :] - rho_e)))
    print("cfg1 L1(rho) vs exact: gpu %.4e oracle %.4e" % (l1, l1_oracle))
    assert l1 <= 1.5e-3 and abs(l1 - l1_oracle) <= 1e-5             # first-order capture of three waves on 1024 cells
    vel = U[1, 3, 5, :] / rho
    P = (G - 1) * (U[4, 3, 5, :] - 0.5 * rho * vel * vel)
    starL = (xi > gold["raref_tail"] + 0.2) & (xi < gold["u_star"] - 0.35)
    starR = (xi > gold["u_star"] + 0.3) & (xi < gold["shock_speed"] - 0.25)
    assert starL.sum() >= 8 and starR.sum() >= 8
    assert np.allclose(rho[starL], gold["rho_star_L"], rtol=1e-2) and np.allclose(rho[starR], gold["rho_star_R"], rtol=1e-2)
    for m in (starL, starR):
        assert np.allclose(P[m], gold["p_star"], rtol=1e-2) and np.allclose(vel[m], gold["u_star"], rtol=1e-2)
    assert rho.max() <= 1.0 + 1e-6 and rho.min() >= 0.125 - 1e-6    # no new extrema


def test_cfg2_turbulence_256_cubed_4096_groups_10_steps():
    """configs[2] as stated: 256^3 periodic, 4096 groups, van Leer, 10 steps at C = 0.5, fp32: oracle parity after
    one step (1e-4, every group, boundary fluxes too) and after ten (1e-3), conservation (P10), guard count 0."""
    w = wl.config_2_turbulence(256, seed=2, steps=10)
    dx = pu.f32(w.dx)
    grp = w.groups()
    assert grp.shape[0] == 4096
    # one step through the plain step call: U_out and boundary fluxes element by element
    gm = []
    out, bf, st = pu.run_gpu(grp, w.dt(), dx, G, w.limiter, guard_map=gm)
    res = pu.compare(grp, w.dt(), dx, G, w.limiter, out, bf, gpu_guard=gm[0])
    print("cfg2 one step: err %.3e bflux %.3e" % (res["err"], res["err_bflux"]))
    assert res["err"] <= 1e-4 and res["err_bflux"] <= 1e-3 and res["excluded_fraction"] == 0.0
    assert st == (0, 0) and res["oracle"].guard_cells == 0
    del out, bf, res, gm
    # ten device-resident steps
    run = DeviceRun(w, np.float32)
    run.advance(10)
    Ug = run.box()
    Uo = _oracle_advance(w.U.astype(np.float64), w, run.dts, dx)
    err = metrics.max_rel_err(Ug[None], Uo[None], G)
    print("cfg2 ten steps: err %.3e" % err)
    assert err <= 1e-3, err
    for q in range(5):                                              # P10: fp32 state, fp64 accumulation
        s0, s1 = w.U[q].astype(np.float64).sum(), Ug[q].astype(np.float64).sum()
        assert abs(s1 - s0) <= 1e-5 * np.abs(w.U[q]).astype(np.float64).sum(), q
    assert gh.gamer_hydro_status() == (0, 0)


@pytest.mark.parametrize("dtype", [np.float64, np.float32])
def test_cfg4_sedov_256_cubed_4096_groups_100_steps(dtype):
    """configs[4] as stated: 256^3 periodic, 4096 groups, MinMod, 100 steps at C = 0.4: positivity of rho and P after
    every step (checked on the device), the Sedov-Taylor radius and exponent of pin P15, and in fp64 parity with the
    oracle on all 4096 groups at step 1 (1e-11) and on the box at step 20."""
    w = wl.config_4_sedov(256, steps=100, dtype=dtype)
    xi0 = _golden("sedov_xi0.txt")["gamma_5_3"]
    n = 256
    run = DeviceRun(w, dtype)
    c = (torch.arange(n, device=DEV, dtype=torch.float64) + 0.5) / n - 0.5
    # radius of every interior cell, in the [G][16][16][16] layout of U_out
    gx = n // 16
    gidx = torch.arange(gx ** 3, device=DEV)
    bx, by, bz = gidx % gx, (gidx // gx) % gx, gidx // (gx * gx)
    o = torch.arange(16, device=DEV)
    X = c[(bx[:, None] * 16 + o[None, :])][:, None, None, :]
    Y = c[(by[:, None] * 16 + o[None, :])][:, None, :, None]
    Z = c[(bz[:, None] * 16 + o[None, :])][:, :, None, None]
    R = torch.sqrt(X * X + Y * Y + Z * Z)
    radii, times, t = [], [], 0.0
    Uo = w.U.astype(np.float64) if dtype == np.float64 else None
    for s in range(100):
        run.advance(1)
        t += run.dts[-1]
        U = run.d_out.double()
        assert float(U[:, 0].min()) > 0
        P = (G - 1) * (U[:, 4] - 0.5 * (U[:, 1] ** 2 + U[:, 2] ** 2 + U[:, 3] ** 2) / U[:, 0])
        assert float(P.min()) > 0, (np.dtype(dtype).name, s, float(P.min()))
        if s + 1 >= 50:
            shell = U[:, 0] > 1.5
            radii.append(float(R[shell].max()) if bool(shell.any()) else 0.0)
            times.append(t)
        if Uo is not None and s < 20:
            Uo = _oracle_advance(Uo, w, [run.dts[-1]], run.dx)
            if s == 0:                                              # every cell of all 4096 groups after one step
                e1 = metrics.max_rel_err(run.box()[None], Uo[None], G)
                print("cfg4 fp64 step 1: err %.3e" % e1)
                assert e1 <= 1e-11, e1
            if s == 19:
                e20 = metrics.max_rel_err(run.box()[None], Uo[None], G)
                print("cfg4 fp64 step 20: err %.3e" % e20)
                assert e20 <= 1e-9, e20
    R_st = xi0 * (w.meta["E0"] * t * t / 1.0) ** 0.2
    print("cfg4 %s: R_num %.5f R_ST %.5f" % (np.dtype(dtype).name, radii[-1], R_st))
    assert abs(radii[-1] - R_st) <= max(1.5 * w.dx, 0.15 * R_st), (radii[-1], R_st)
    slope = np.polyfit(np.log(times), np.log(radii), 1)[0]
    assert 0.34 <= slope <= 0.46, slope
