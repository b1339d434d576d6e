"""Pins P1–P16 of SURVEY.md §8(c): the fp64 oracle checked against what the mathematics fixes — closed
forms, identities, exact solutions, brute force — never against itself and never against the CUDA path.
PAPER.md prints no worked example, so there are no paper values to store; tests/golden/ holds the
mathematical constants (exact Sod star state, Sedov xi0) with their provenance. All CPU, `-m "not gpu"`."""
import math
import os

import numpy as np
import pytest

import exact_riemann as er
import naive_mhm
from oracle import mhm_oracle as O
from harness import workloads as wl

G = 5.0 / 3.0
HERE = os.path.dirname(os.path.abspath(__file__))


def cons(rho, vx, vy, vz, P, g=G):
    return np.array([rho, rho * vx, rho * vy, rho * vz, P / (g - 1) + 0.5 * rho * (vx * vx + vy * vy + vz * vz)])


def closed_form_flux(rho, vx, vy, vz, P, d, g=G):
    """F_d(U) written out from the Euler equations (not via the oracle)."""
    v = (vx, vy, vz)
    E = P / (g - 1) + 0.5 * rho * (vx * vx + vy * vy + vz * vz)
    F = np.array([rho * v[d], rho * vx * v[d], rho * vy * v[d], rho * vz * v[d], (E + P) * v[d]])
    F[1 + d] += P
    return F


def random_states(n, seed):
    rng = np.random.default_rng(seed)
    out = []
    for _ in range(n):
        out.append(cons(rng.uniform(0.1, 10), *rng.normal(0, 2, 3), rng.uniform(0.01, 10)))
    return out


def read_golden(name):
    d = {}
    for line in open(os.path.join(HERE, "golden", name)):
        if line.strip() and not line.startswith("#"):
            k, v = line.split()
            d[k] = float(v)
    return d


# ---------------------------------------------------------------- O1/O4 building blocks vs closed forms


def test_variable_set_roundtrip_and_flux_closed_form():
    rng = np.random.default_rng(5)
    for _ in range(200):
        W = np.array([rng.uniform(0.1, 10), *rng.normal(0, 2, 3), rng.uniform(0.01, 10)])
        U = O.prim_to_cons(W, G)
        assert np.allclose(U, cons(*W), rtol=1e-15, atol=0)
        assert np.allclose(O.cons_to_prim(U, G), W, rtol=1e-12, atol=1e-13)
        for d in range(3):
            assert np.allclose(O.phys_flux(U, G, d), closed_form_flux(*W, d), rtol=1e-13, atol=1e-13)


# ---------------------------------------------------------------- P1


@pytest.mark.parametrize("d", [0, 1, 2])
def test_P1_roe_consistency_bit_exact(d):
    for U in random_states(500, 11):
        assert np.array_equal(O.roe_flux(U, U, G, d), O.phys_flux(U, G, d))


# ---------------------------------------------------------------- P2


@pytest.mark.parametrize("limiter", [0, 1])
def test_P2_uniform_moving_state_preserved_bit_exact(limiter):
    W = (1.3, 0.37, -0.61, 0.23, 0.9)
    U = cons(*W)
    N, S = 16, 20
    Uin = np.broadcast_to(U[:, None, None, None], (2, 5, S, S, S)).copy()
    r = O.step_groups(Uin, N, 2, 0.004, 1.0 / 32, G, limiter)
    assert np.array_equal(r.U_out, Uin[:, :, 2:-2, 2:-2, 2:-2])
    assert r.guard_cells == 0 and r.nonpositive_out == 0
    for f in range(6):
        Fd = closed_form_flux(*W, f // 2)
        assert np.allclose(r.bflux[:, f], Fd[None, :, None, None], rtol=1e-13, atol=1e-14)


# ---------------------------------------------------------------- P3


@pytest.mark.parametrize("d", [0, 1, 2])
def test_P3_roe_identities(d):
    n, t1, t2 = d, (d + 1) % 3, (d + 2) % 3
    rot = [0, 1 + n, 1 + t1, 1 + t2, 4]
    S = random_states(2000, 21 + d)
    worst = 0.0
    for UL, UR in zip(S[::2], S[1::2]):
        al, lam, K = O.roe_decompose(UL, UR, G, d)
        dU = (UR - UL)[rot]
        WL = O.cons_to_prim(UL, G)
        WR = O.cons_to_prim(UR, G)
        dF = (closed_form_flux(*WR, d) - closed_form_flux(*WL, d))[rot]
        e1 = np.abs(al @ K - dU).max() / np.abs(dU).max()
        e2 = np.abs((al * lam) @ K - dF).max() / max(np.abs(dF).max(), np.abs(lam).max() * np.abs(dU).max())
        worst = max(worst, e1, e2)
        # flux = central average minus half the |lambda|-weighted decomposition (definition of Roe's flux)
        F = O.roe_flux(UL, UR, G, d)[rot]
        Fdef = 0.5 * (closed_form_flux(*WL, d) + closed_form_flux(*WR, d))[rot] - 0.5 * (al * np.abs(lam)) @ K
        assert np.allclose(F, Fdef, rtol=1e-11, atol=1e-11)
    assert worst <= 1e-12, worst


def test_P3b_roe_strengths_equal_primitive_jump_form():
    """alpha_1,5 = (dp -+ rho~ a~ du)/(2a~^2), alpha_2 = drho - dp/a~^2, alpha_3,4 = rho~ dv, rho~ dw."""
    S = random_states(2000, 31)
    for UL, UR in zip(S[::2], S[1::2]):
        al, lam, K = O.roe_decompose(UL, UR, G, 0)
        WL, WR = O.cons_to_prim(UL, G), O.cons_to_prim(UR, G)
        a = 0.5 * (lam[4] - lam[0])
        rt = math.sqrt(WL[0] * WR[0])
        d = WR - WL
        b = np.array([(d[4] - rt * a * d[1]) / (2 * a * a), d[0] - d[4] / (a * a), rt * d[2], rt * d[3],
                      (d[4] + rt * a * d[1]) / (2 * a * a)])
        assert np.abs(b - al).max() <= 1e-10 * max(1.0, np.abs(al).max())


# ---------------------------------------------------------------- P4


@pytest.mark.parametrize("d", [0, 1, 2])
def test_P4_supersonic_upwinding(d):
    rng = np.random.default_rng(41)
    for sign in (+1, -1):
        for _ in range(200):
            v = rng.normal(0, 0.3, 3)
            WL = [rng.uniform(0.5, 2), *v, rng.uniform(0.5, 2)]
            WR = [rng.uniform(0.5, 2), *(v + rng.normal(0, 0.1, 3)), rng.uniform(0.5, 2)]
            WL[1 + d] = sign * rng.uniform(8, 12)   # |u| >> a on both sides => all eigenvalues share the sign
            WR[1 + d] = sign * rng.uniform(8, 12)
            UL, UR = cons(*WL), cons(*WR)
            al, lam, K = O.roe_decompose(UL, UR, G, d)
            assert np.all(sign * lam > 0)
            F = O.roe_flux(UL, UR, G, d)
            Fup = closed_form_flux(*(WL if sign > 0 else WR), d)
            assert np.allclose(F, Fup, rtol=1e-11, atol=1e-11)


# ---------------------------------------------------------------- P5


def _stationary_shock(M1=3.0, g=G):
    """Rankine–Hugoniot pair in the shock frame: upstream (rho1,u1,p1) with Mach M1, downstream from the jump
    conditions; F(UL) = F(UR) exactly in exact arithmetic."""
    r1, p1 = 1.0, 1.0
    u1 = M1 * math.sqrt(g * p1 / r1)
    r2 = r1 * (g + 1) * M1 * M1 / ((g - 1) * M1 * M1 + 2)
    p2 = p1 * (2 * g * M1 * M1 - (g - 1)) / (g + 1)
    u2 = u1 * r1 / r2
    return (r1, u1, p1), (r2, u2, p2)


@pytest.mark.parametrize("d", [0, 1, 2])
def test_P5_stationary_shock_and_contact_flux(d):
    (r1, u1, p1), (r2, u2, p2) = _stationary_shock()
    vL, vR = [0.2, -0.1, 0.3], [0.2, -0.1, 0.3]  # transverse velocity continuous across a shock
    vL[d], vR[d] = u1, u2
    UL, UR = cons(r1, *vL, p1), cons(r2, *vR, p2)
    F = O.roe_flux(UL, UR, G, d)
    FL = closed_form_flux(r1, *vL, p1, d)
    assert np.allclose(F, FL, rtol=1e-12, atol=1e-12)
    # stationary contact: rho jump, u = 0 along d, equal p, (a shear in the transverse velocity is allowed)
    vL, vR = [0.3, 0.3, 0.3], [-0.4, -0.4, -0.4]
    vL[d] = vR[d] = 0.0
    UL, UR = cons(2.0, *vL, 0.7), cons(0.5, *vR, 0.7)
    F = O.roe_flux(UL, UR, G, d)
    expect = np.zeros(5)
    expect[1 + d] = 0.7
    assert np.allclose(F, expect, rtol=0, atol=1e-15)


def test_P5_stationary_contact_stays_exactly_stationary_many_steps():
    nx = 32
    rho = np.where(np.arange(nx) < nx // 2, 2.0, 0.5)
    rho = np.broadcast_to(rho[None, None, :], (16, 16, nx))
    z = np.zeros_like(rho)
    U0 = wl.prim_box_to_cons(rho, z, z, z, 0.7 + z)
    step = lambda grp, dt: O.step_groups(grp, 16, 2, dt, 1.0 / nx, G, 0, want_bflux=False, want_guard=False).U_out
    U, t, dts = wl.advance(U0, 1.0 / nx, ("outflow", "periodic", "periodic"), 0, 0.5, 20, step, dtype=np.float64)
    assert np.array_equal(U[0], U0[0])            # density profile untouched
    assert np.array_equal(U[1:4], U0[1:4])        # still at rest, exactly
    assert np.allclose(U[4], U0[4], rtol=1e-15)


# ---------------------------------------------------------------- P6


@pytest.mark.parametrize("axis", [0, 1, 2])
def test_P6_moving_contact_hand_value(axis):
    """rho step 1 -> 2, u = 1 along `axis`, P = 1, MinMod, lambda = dt/dx = 0.25: slopes vanish at the step,
    Roe reduces to donor cell, so the first cell right of the step becomes 2 - 0.25 (2 - 1) = 1.75; u, P unchanged."""
    n = 32
    dims = [16, 16, 16]
    dims[axis] = n
    nx, ny, nz = dims
    prof = np.where(np.arange(n) < n // 2, 1.0, 2.0)
    shp = [1, 1, 1]
    shp[2 - axis] = n
    rho = np.broadcast_to(prof.reshape(shp), (nz, ny, nx))
    v = [np.zeros((nz, ny, nx)) for _ in range(3)]
    v[axis] = v[axis] + 1.0
    U0 = wl.prim_box_to_cons(rho, *v, np.ones((nz, ny, nx)))
    bc = ["periodic"] * 3
    bc[axis] = "outflow"
    dx = 1.0 / n
    r = O.step_groups(wl.cut_groups(U0, bc), 16, 2, 0.25 * dx, dx, G, 0)
    U1 = wl.assemble_box(r.U_out, (nz, ny, nx))
    rho1 = np.moveaxis(U1[0], 2 - axis, 0)[:, 0, 0]
    expect = prof.copy()
    expect[n // 2] = 1.75
    assert np.allclose(rho1, expect, rtol=0, atol=1e-14), rho1
    W = np.array([O.cons_to_prim(U1[:, 3, 5, i] if axis == 0 else (U1[:, 3, i, 5] if axis == 1 else U1[:, i, 3, 5]), G)
                  for i in range(n)])
    assert np.allclose(W[:, 1 + axis], 1.0, atol=1e-14)
    assert np.allclose(W[:, 4], 1.0, atol=1e-13)
    other = [1 + a for a in range(3) if a != axis]
    assert np.all(W[:, other] == 0.0)


# ---------------------------------------------------------------- P7


@pytest.mark.parametrize("limiter", [0, 1])
def test_P7_limiters_on_linear_field_and_extrema(limiter):
    for b in (0.25, -1.5, 3.0, 1e-7):
        if limiter == 0:
            assert O.limited_slope(b, b, limiter) == b      # linear field: exactly b dx
        else:                                               # 2 b b / (b + b): b*b rounds once
            assert O.limited_slope(b, b, limiter) == pytest.approx(b, rel=4e-16)
    assert O.limited_slope(1.0, -2.0, limiter) == 0.0       # local extremum
    assert O.limited_slope(-1.0, 2.0, limiter) == 0.0
    assert O.limited_slope(0.0, 2.0, limiter) == 0.0        # zero included
    assert O.limited_slope(2.0, 0.0, limiter) == 0.0
    assert O.limited_slope(1e-200, -1e-200, limiter) == 0.0  # sign test does not underflow
    if limiter == 0:    # (the van Leer quotient 2 dL dR/(dL+dR) itself underflows to 0 here, harmlessly)
        assert O.limited_slope(1e-200, 3e-200, limiter) == 1e-200
    # textbook values
    if limiter == 0:
        assert O.limited_slope(1.0, 3.0, 0) == 1.0 and O.limited_slope(-4.0, -3.0, 0) == -3.0
    else:
        assert O.limited_slope(1.0, 3.0, 1) == pytest.approx(1.5, rel=1e-15)      # 2*1*3/4
        assert O.limited_slope(-4.0, -2.0, 1) == pytest.approx(-8.0 / 3.0, rel=1e-15)
    # symmetry and the bound |slope| <= 2 min(|dL|,|dR|) used in O3's positivity argument
    rng = np.random.default_rng(7)
    for dL, dR in rng.normal(0, 1, (500, 2)):
        s = O.limited_slope(dL, dR, limiter)
        assert s == O.limited_slope(dR, dL, limiter)
        assert O.limited_slope(-dL, -dR, limiter) == -s
        assert abs(s) <= 2 * min(abs(dL), abs(dR)) * (1 + 1e-15)


# ---------------------------------------------------------------- P8


def _entropy_wave(n, nvec, steps_per_period_frac=0.25, limiter=1):
    """rho = 1 + 0.2 sin(2 pi n.x), uniform v and P, periodic; advect for a fixed time; return L1 error of rho."""
    dx = 1.0 / n
    c = (np.arange(n) + 0.5) * dx
    Z, Y, X = np.meshgrid(c, c, c, indexing="ij")
    v = np.array([0.9, 0.6, 0.3])
    phase = lambda t: 2 * math.pi * (nvec[0] * (X - v[0] * t) + nvec[1] * (Y - v[1] * t) + nvec[2] * (Z - v[2] * t))
    rho0 = 1 + 0.2 * np.sin(phase(0.0))
    one = np.ones_like(rho0)
    U = wl.prim_box_to_cons(rho0, v[0] * one, v[1] * one, v[2] * one, one)
    T = 0.05
    cmax = wl.max_signal_speed(U)
    nsteps = int(math.ceil(T / (0.4 * dx / cmax)))
    dt = T / nsteps
    for _ in range(nsteps):
        r = O.step_groups(wl.cut_groups(U, ("periodic",) * 3), 16, 2, dt, dx, G, limiter, want_bflux=False,
                          want_guard=False)
        U = wl.assemble_box(r.U_out, (n, n, n))
    return float(np.mean(np.abs(U[0] - (1 + 0.2 * np.sin(phase(T))))))


@pytest.mark.parametrize("nvec", [(1, 0, 0), (1, 1, 1)])
def test_P8_second_order_convergence_entropy_wave(nvec):
    e16, e32 = _entropy_wave(16, nvec), _entropy_wave(32, nvec)
    assert e16 / e32 >= 3.3, (e16, e32, e16 / e32)


# ---------------------------------------------------------------- P9


def test_exact_riemann_solver_matches_golden_constants():
    gold = read_golden("sod_exact_gamma53.txt")
    mine = er.sod_constants(G)
    for k, v in gold.items():
        assert mine[k] == pytest.approx(v, rel=2e-9), k
    ps, us = er.star_state(1.4, 1, 0, 1, 0.125, 0, 0.1)     # textbook check of the solver itself
    assert ps == pytest.approx(0.30313, abs=1e-5) and us == pytest.approx(0.92745, abs=1e-5)


def _sod_run(nx, limiter=0, axis=0, reverse=False):
    w = wl.config_1_sod_tube(nx=nx, limiter=limiter, steps=200 * nx // 1024, axis=axis, reverse=reverse,
                             dtype=np.float64)
    step = lambda grp, dt: O.step_groups(grp, 16, 2, dt, w.dx, G, limiter, want_bflux=False, want_guard=False).U_out
    U, t, dts = wl.advance(w.U, w.dx, w.bc, limiter, w.cfl, w.steps, step, dtype=np.float64)
    return w, U, t


def test_P9_sod_tube_vs_exact_solution():
    gold = read_golden("sod_exact_gamma53.txt")
    errs = {}
    for nx in (512, 1024):
        w, U, t = _sod_run(nx)
        x = (np.arange(nx) + 0.5) / nx
        rho_e, u_e, p_e = er.sample(G, (1, 0, 1), (0.125, 0, 0.1), (x - 0.5) / t)
        rho = U[0, 3, 5, :]
        errs[nx] = float(np.mean(np.abs(rho - rho_e)))
        assert np.array_equal(U[2], np.zeros_like(U[2])) and np.array_equal(U[3], np.zeros_like(U[3]))
        assert np.array_equal(U[:, 3, 5, :], U[:, 11, 2, :])       # stays 1-D
        if nx == 1024:     # configs[1] proper: 64 groups, 200 steps
            W = np.array([O.cons_to_prim(U[:, 3, 5, i], G) for i in range(nx)])
            xi = (x - 0.5) / t
            # plateaus between the waves, away from the smeared transitions
            starL = (xi > gold["raref_tail"] + 0.2) & (xi < gold["u_star"] - 0.35)
            starR = (xi > gold["u_star"] + 0.3) & (xi < gold["shock_speed"] - 0.25)
            assert starL.sum() >= 8 and starR.sum() >= 8
            assert np.allclose(W[starL, 0], gold["rho_star_L"], rtol=1e-2)
            assert np.allclose(W[starR, 0], gold["rho_star_R"], rtol=1e-2)
            for m in (starL, starR):
                assert np.allclose(W[m, 4], gold["p_star"], rtol=1e-2)
                assert np.allclose(W[m, 1], gold["u_star"], rtol=1e-2)
            assert rho.max() <= 1.0 + 1e-12 and rho.min() >= 0.125 - 1e-12   # no new extrema
    ratio = errs[512] / errs[1024]
    assert 1.5 <= ratio <= 2.6, (errs, ratio)    # about first order for a solution with discontinuities


# ---------------------------------------------------------------- P10 / P11 / P12


def test_P10_global_conservation_periodic():
    w = wl.config_2_turbulence(32, seed=7)
    U0 = w.U.astype(np.float64)
    step = lambda grp, dt: O.step_groups(grp, 16, 2, dt, w.dx, G, w.limiter, want_bflux=False, want_guard=False).U_out
    U, t, dts = wl.advance(U0, w.dx, w.bc, w.limiter, w.cfl, 5, step, dtype=np.float64)
    assert np.abs(U - U0).max() > 1e-4   # something happened
    for q in range(5):
        s0, s1 = U0[q].sum(), U[q].sum()
        scale = np.abs(U0[q]).sum()
        assert abs(s1 - s0) <= 1e-12 * scale, (q, s0, s1)


def test_P11_group_balance_and_face_layout():
    w = wl.config_2_turbulence(32, seed=8)
    grp = w.groups(np.float64)
    dt = w.dt()
    r = O.step_groups(grp, 16, 2, dt, w.dx, G, w.limiter)
    lam = dt / w.dx
    dU = (r.U_out - grp[:, :, 2:-2, 2:-2, 2:-2]).sum(axis=(2, 3, 4))               # [G,5]
    net = sum(r.bflux[:, 2 * d + 1].sum(axis=(2, 3)) - r.bflux[:, 2 * d].sum(axis=(2, 3)) for d in range(3))
    scale = np.abs(grp[:, :, 2:-2, 2:-2, 2:-2]).sum(axis=(2, 3, 4))
    assert np.all(np.abs(dU + lam * net) <= 1e-13 * scale)
    # neighbouring groups share faces: +x flux of group g equals -x flux of its x-neighbour, bit for bit
    b = r.bflux.reshape(2, 2, 2, 6, 5, 16, 16)
    assert np.array_equal(b[:, :, 0, 1], b[:, :, 1, 0]) and np.array_equal(b[:, :, 1, 1], b[:, :, 0, 0])
    assert np.array_equal(b[:, 0, :, 3], b[:, 1, :, 2]) and np.array_equal(b[0, :, :, 5], b[1, :, :, 4])
    # a single hot cell next to one face pins face order and in-face index order (lower axis fastest)
    S = 20
    base = cons(1.0, 0, 0, 0, 1.0)
    for face, (i, j, k) in {0: (0, 5, 9), 1: (15, 5, 9), 2: (5, 0, 9), 3: (5, 15, 9), 4: (5, 9, 0), 5: (5, 9, 15)}.items():
        Uin = np.broadcast_to(base[:, None, None, None], (1, 5, S, S, S)).copy()
        Uin[0, 4, k + 2, j + 2, i + 2] *= 3.0      # hot cell (pressure x3), interior index (i,j,k)
        rr = O.step_groups(Uin, 16, 2, 1e-3, 1.0 / 16, G, 0)
        rest = np.broadcast_to(closed_form_flux(1.0, 0, 0, 0, 1.0, face // 2)[:, None, None], (5, 16, 16))
        dev = np.abs(rr.bflux[0, face] - rest).sum(axis=0)     # [16][16]
        a, b2 = np.unravel_index(np.argmax(dev), dev.shape)
        inface = {0: (k, j), 1: (k, j), 2: (k, i), 3: (k, i), 4: (j, i), 5: (j, i)}[face]
        assert (a, b2) == inface, (face, a, b2)
        for other in range(6):
            if other != face:
                rest_o = closed_form_flux(1.0, 0, 0, 0, 1.0, other // 2)
                assert np.abs(rr.bflux[0, other] - rest_o[:, None, None]).max() < dev.max()


@pytest.mark.parametrize("bc", [("periodic",) * 3, ("outflow", "periodic", "outflow")])
def test_P12_decomposition_invariance_bit_identical(bc):
    w = wl.config_2_turbulence(32, seed=9)
    U0 = w.U.astype(np.float64)
    dt = w.dt()
    per_group = wl.assemble_box(O.step_groups(wl.cut_groups(U0, bc), 16, 2, dt, w.dx, G, 1).U_out, (32, 32, 32))
    whole = O.step_box(wl.pad_box(U0, bc), 2, dt, w.dx, G, 1).U_out
    assert np.array_equal(per_group, whole)


def test_ghost_width_3_reads_only_two_layers():
    g2 = wl.random_groups(2, seed=5, ghost=2, dtype=np.float64)
    g3 = np.full((2, 5, 22, 22, 22), np.nan)
    g3[:, :, 1:-1, 1:-1, 1:-1] = g2
    a = O.step_groups(g2, 16, 2, 1e-3, 1 / 16, G, 0)
    b = O.step_groups(g3, 16, 3, 1e-3, 1 / 16, G, 0)
    assert np.array_equal(a.U_out, b.U_out) and np.array_equal(a.bflux, b.bflux)


def test_unneeded_ghost_cells_are_never_read():
    """The 640 corner / layer-2 edge ghosts of a 20^3 group are outside the five-point stencil."""
    g = wl.random_groups(1, seed=6, dtype=np.float64)
    a = O.step_groups(g, 16, 2, 1e-3, 1 / 16, G, 1)
    h = g.copy()
    idx = np.arange(20)
    depth = np.where(idx < 2, 2 - idx, np.where(idx > 17, idx - 17, 0))
    tot = depth[:, None, None] + depth[None, :, None] + depth[None, None, :]
    assert (tot > 2).sum() == 640
    h[:, :, tot > 2] = np.nan
    b = O.step_groups(h, 16, 2, 1e-3, 1 / 16, G, 1)
    assert np.array_equal(a.U_out, b.U_out) and np.array_equal(a.bflux, b.bflux)


# ---------------------------------------------------------------- P13


def _reflect(grp, axis):
    """Mirror a batch [G,5,S,S,S] about the plane normal to `axis` (0=x) and negate that momentum."""
    out = np.flip(grp, axis=4 - axis).copy()
    out[:, 1 + axis] *= -1.0
    return out


@pytest.mark.parametrize("limiter", [0, 1])
@pytest.mark.parametrize("axis", [0, 1, 2])
def test_P13_mirror_symmetry_bit_exact(axis, limiter):
    g = wl.random_groups(2, seed=13, dtype=np.float64)
    a = O.step_groups(g, 16, 2, 2e-3, 1 / 16, G, limiter)
    b = O.step_groups(_reflect(g, axis), 16, 2, 2e-3, 1 / 16, G, limiter)
    assert np.array_equal(_reflect(a.U_out, axis), b.U_out)


def test_P13_axis_permutation_roundoff():
    g = wl.random_groups(1, seed=14, dtype=np.float64)
    a = O.step_groups(g, 16, 2, 2e-3, 1 / 16, G, 1).U_out
    # cyclic relabelling x->y->z->x: new array index order [z'][y'][x'] = [y][x][z], momenta permuted alike
    p = np.transpose(g, (0, 1, 3, 4, 2))[:, [0, 3, 1, 2, 4]].copy()
    b = O.step_groups(p, 16, 2, 2e-3, 1 / 16, G, 1).U_out
    back = np.transpose(b[:, [0, 2, 3, 1, 4]], (0, 1, 4, 2, 3))
    assert np.allclose(back, a, rtol=1e-12, atol=1e-13)


def test_P13_sod_along_every_axis_and_direction():
    ref = None
    for axis in (0, 1, 2):
        for reverse in (False, True):
            w, U, t = _sod_run(64, axis=axis, reverse=reverse)
            prof = np.moveaxis(U[0], 2 - axis, 0)[:, 0, 0]
            if reverse:
                prof = prof[::-1]
            if ref is None:
                ref = prof
            else:
                assert np.allclose(prof, ref, rtol=1e-12, atol=1e-13), (axis, reverse)


# ---------------------------------------------------------------- P14


@pytest.mark.parametrize("limiter", [0, 1])
def test_P14_one_dimensional_reduction(limiter):
    nx = 64
    x = (np.arange(nx) + 0.5) / nx
    rho = 1 + 0.3 * np.sin(2 * math.pi * x) + 0.5 * (x > 0.6)
    u = 0.4 * np.cos(2 * math.pi * x)
    p = 1 + 0.2 * np.sin(4 * math.pi * x)
    U1 = np.array([rho, rho * u, p / (G - 1) + 0.5 * rho * u * u])
    b = lambda a: np.broadcast_to(a[None, None, :], (16, 16, nx))
    U3 = wl.prim_box_to_cons(b(rho), b(u), b(0 * x), b(0 * x), b(p))
    dx = 1.0 / nx
    for _ in range(5):
        dt = wl.cfl_dt(U3, dx, 0.5)
        U1 = naive_mhm.mhm_1d(U1, dt, dx, G, limiter, "periodic")
        r = O.step_groups(wl.cut_groups(U3, ("periodic",) * 3), 16, 2, dt, dx, G, limiter, want_bflux=False)
        U3 = wl.assemble_box(r.U_out, (16, 16, nx))
    assert np.allclose(U3[[0, 1, 4], 7, 3, :], U1, rtol=1e-12, atol=1e-13)
    assert np.all(U3[2] == 0) and np.all(U3[3] == 0)


# ---------------------------------------------------------------- P15 (scaled-down; the 256^3 run is a gpu test)


def test_P15_sedov_blast_radius_and_positivity():
    xi0 = read_golden("sedov_xi0.txt")["gamma_5_3"]
    n = 64
    w = wl.config_4_sedov(n, steps=100)
    radii, times = [], []
    c = (np.arange(n) + 0.5) / n - 0.5
    R = np.sqrt(c[:, None, None] ** 2 + c[None, :, None] ** 2 + c[None, None, :] ** 2)

    def on_step(i, U, t):
        assert U[0].min() > 0
        P = (G - 1) * (U[4] - 0.5 * (U[1] ** 2 + U[2] ** 2 + U[3] ** 2) / U[0])
        assert P.min() > 0, (i, P.min())
        if i + 1 >= 50:
            # shock radius: density-jump-weighted mean radius of the compressed shell's outer edge
            shell = U[0] > 1.5
            radii.append(R[shell].max() if shell.any() else 0.0)
            times.append(t)

    step = lambda grp, dt: O.step_groups(grp, 16, 2, dt, w.dx, G, 0, want_bflux=False, want_guard=False).U_out
    U, t, dts = wl.advance(w.U, w.dx, w.bc, 0, w.cfl, w.steps, step, dtype=np.float64, on_step=on_step)
    R_st = xi0 * (w.meta["E0"] * t * t / 1.0) ** 0.2
    assert abs(radii[-1] - R_st) <= max(1.5 * w.dx, 0.15 * R_st), (radii[-1], R_st)
    slope = np.polyfit(np.log(times), np.log(radii), 1)[0]
    assert 0.34 <= slope <= 0.46, slope


# ---------------------------------------------------------------- P16


@pytest.mark.parametrize("limiter", [0, 1])
def test_P16_brute_force_second_transcription(limiter):
    g = wl.random_groups(3, seed=16, dtype=np.float64)
    dt, dx = 2e-3, 1 / 16
    r = O.step_groups(g, 16, 2, dt, dx, G, limiter)
    for n in range(3):
        out, bf, guard = naive_mhm.step_group_naive(g[n], 16, 2, dt, dx, G, limiter)
        assert np.allclose(out, r.U_out[n], rtol=1e-11, atol=1e-12)
        assert np.allclose(bf, r.bflux[n], rtol=1e-10, atol=1e-11)
    # tiny group, N = 4, ghost = 2
    g4 = wl.random_groups(2, seed=17, N=4, dtype=np.float64)
    r4 = O.step_groups(g4, 4, 2, dt, dx, G, limiter)
    for n in range(2):
        out, bf, guard = naive_mhm.step_group_naive(g4[n], 4, 2, dt, dx, G, limiter)
        assert np.allclose(out, r4.U_out[n], rtol=1e-11, atol=1e-12)
        assert np.allclose(bf, r4.bflux[n], rtol=1e-10, atol=1e-11)


def test_guard_rule_fallback_is_first_order_and_counted():
    """R7 (parity unpinned: a convention). What can be checked: when the guard fires the cell's six face
    states fall back to its own input state, the event is counted, and both transcriptions agree on where."""
    w = wl.config_3_cosmo(32, seed=3)
    grp = w.groups(np.float64)
    dt = w.dt()
    r = O.step_groups(grp, 16, 2, dt, w.dx, G, 0)
    assert r.guard_cells > 0 and r.guard_cells == int(r.guard.sum())
    n_checked = 0
    for n in range(grp.shape[0]):
        out, bf, guard = naive_mhm.step_group_naive(grp[n], 16, 2, dt, w.dx, G, 0)
        idx = np.arange(18)
        ghost = ((idx == 0) | (idx == 17)).astype(int)
        inR = (ghost[:, None, None] + ghost[None, :, None] + ghost[None, None, :]) <= 1
        near = np.abs(r.margin[n]) < 1e-9
        assert np.array_equal(guard[inR & ~near], r.guard[n][inR & ~near].astype(bool))
        if not near[inR].any():
            e = np.abs(out - r.U_out[n]) / (np.abs(r.U_out[n]) + np.abs(out).max(axis=(1, 2, 3), keepdims=True) * 1e-3)
            assert e.max() < 1e-9
            n_checked += 1
    assert n_checked >= 4


def test_flop_tally_band():
    """The CountingReal tally (the roofline numerator) stays inside the hand-count band of SURVEY.md App. D."""
    S = 20
    z, y, x = np.meshgrid(*(np.arange(S, dtype=np.float64),) * 3, indexing="ij")
    ramp = 1.0 + 0.01 * (x + 2 * y + 3 * z)          # every slope active (monotone in all directions)
    U = wl.prim_box_to_cons(ramp, 0.1 * ramp, -0.2 * ramp, 0.3 * ramp, 2.0 * ramp)
    c0 = O.count_flops(U, 16, 2, 1e-3, 1 / 16, G, 0)
    c1 = O.count_flops(U, 16, 2, 1e-3, 1 / 16, G, 1)
    assert 0.85 * 925 <= c0["per_cell"] <= 1.15 * 925, c0
    assert c1["per_cell"] > c0["per_cell"]
    assert c0["sqrt"] == 3 * 13056 and c0["minmax"] == 15 * 5632


def test_sedov_golden_constants_are_rederived_by_the_committed_calculator():
    """tests/golden/sedov_xi0.txt (used by P15 and the cfg 4 tests for the shock radius) against tests/sedov_taylor.py:
    the self-similar ODEs integrated inward from the strong-shock conditions and normalised by the energy integral
    (SURVEY.md Appendix A). gamma = 1.4 gives the textbook 1.033; a closed form exists for no gamma, but the integrated
    profile must show the flat central pressure of Taylor's solution, P(0) / P(1) = 0.366 for gamma = 1.4."""
    import sedov_taylor as st
    golden = {}
    with open(os.path.join(os.path.dirname(__file__), "golden", "sedov_xi0.txt")) as f:
        for line in f:
            if line.strip() and not line.startswith("#"):
                k, v = line.split()
                golden[k] = float(v)
    assert abs(st.xi0(5.0 / 3.0) - golden["gamma_5_3"]) <= 1e-5
    assert abs(st.xi0(1.4) - golden["gamma_1_4"]) <= 1e-5
    assert abs(st.xi0(1.4) - 1.033) <= 5e-4                              # the value every textbook prints
    assert abs(st.xi0(1.4, lam_min=1e-2) - st.xi0(1.4, lam_min=1e-4)) <= 1e-9   # the inner cut-off does not matter
    sol = st.profiles(1.4)
    assert abs(np.exp(sol.y[2, -1] - sol.y[2, 0]) - 0.366) <= 2e-3       # central over post-shock pressure
    assert sol.y[1, -1] < np.log(1e-6)                                   # the centre is evacuated
