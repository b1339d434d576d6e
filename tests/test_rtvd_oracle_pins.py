"""Pins of the relaxing-TVD oracle (oracle/rtvd_oracle.hpp): closed forms,
invariants, the exact Riemann solution, a whole-array transcription — never the oracle against itself and never against
the CUDA path. All CPU, `-m "not gpu"`."""
import numpy as np
import pytest

import exact_riemann as er
import naive_rtvd
from harness import workloads as wl
from oracle import rtvd_oracle as R

G = 5.0 / 3.0


def cons(rho, vx, vy, vz, P, g=G):
    return np.array([rho, rho * vx, rho * vy, rho * vz, P / (g - 1) + 0.5 * rho * (vx * vx + vy * vy + vz * vz)])


def smooth_box(n, seed, amp=0.2):
    rng = np.random.default_rng(seed)
    c = (np.arange(n) + 0.5) / n
    Z, Y, X = np.meshgrid(c, c, c, indexing="ij")
    ph = rng.uniform(0, 2 * np.pi, 6)
    rho = 1.0 + amp * np.sin(2 * np.pi * X + ph[0]) * np.cos(2 * np.pi * Y + ph[1]) + 0.1 * np.sin(4 * np.pi * Z + ph[2])
    P = 1.0 + amp * np.cos(2 * np.pi * (X + Y + Z) + ph[3])
    vx = 0.5 * np.sin(2 * np.pi * Y + ph[4]); vy = -0.3 * np.cos(2 * np.pi * Z + ph[5]); vz = 0.4 * np.sin(2 * np.pi * X)
    return wl.prim_box_to_cons(rho, vx, vy, vz, P)


@pytest.mark.parametrize("d", [0, 1, 2])
def test_flux_is_the_euler_flux_and_speed_is_v_plus_cs(d):
    rng = np.random.default_rng(3)
    for _ in range(100):
        rho, P = rng.uniform(0.1, 10), rng.uniform(0.01, 10)
        v = rng.normal(0, 2, 3)
        F, c = R.flux_and_speed(cons(rho, *v, P), d, G)
        E = P / (G - 1) + 0.5 * rho * (v @ v)
        want = np.array([rho * v[d], rho * v[0] * v[d], rho * v[1] * v[d], rho * v[2] * v[d], (E + P) * v[d]])
        want[1 + d] += P
        assert np.allclose(F, want, rtol=1e-13, atol=1e-13)
        assert abs(c - (abs(v[d]) + np.sqrt(G * P / rho))) <= 1e-12 * c


def test_vanleer_hand_values():
    assert R.vanleer(1.0, 3.0) == 1.5 and R.vanleer(-1.0, -3.0) == -1.5      # harmonic mean 2ab/(a+b)
    assert R.vanleer(1.0, -3.0) == 0.0 and R.vanleer(0.0, 2.0) == 0.0 and R.vanleer(2.0, 0.0) == 0.0
    assert abs(R.vanleer(1e-100, 1e-100) - 1e-100) <= 1e-115                  # sign test by comparison, not by a product
    for a, b in ((0.3, 0.7), (5.0, 0.01)):                                    # TVD region: 0 <= phi <= 2 min(a, b)
        assert 0.0 <= R.vanleer(a, b) <= 2.0 * min(a, b)


@pytest.mark.parametrize("sweep", [0, 1])
def test_uniform_moving_state_is_preserved_bit_exactly(sweep):
    U = cons(1.3, 0.37, -0.61, 0.23, 0.9)
    box = np.broadcast_to(U[:, None, None, None], (5, 14, 14, 14)).copy()
    out = R.step_box(box, 0.004, 1.0 / 32, G, sweep)
    assert np.array_equal(out, box[:, 3:-3, 3:-3, 3:-3])


@pytest.mark.parametrize("sweep", [0, 1])
def test_whole_box_array_shift_transcription(sweep):
    """Brute force: the oracle's line loops with 3 ghost cells against a whole-array periodic transcription."""
    n = 16
    U = smooth_box(n, 5)
    dt, dx = 0.2 / n / 3.0, 1.0 / n
    out = R.step_box(wl.pad_box(U, ("periodic",) * 3, 3), dt, dx, G, sweep)
    want = naive_rtvd.step_periodic(U, dt, dx, G, sweep)
    assert np.abs(out - want).max() <= 1e-14 * np.abs(want).max()
    assert np.abs(out - U).max() > 1e-4                                       # something happened
    # and the two sweep orders differ (the splitting error), so `sweep` is really honoured
    other = R.step_box(wl.pad_box(U, ("periodic",) * 3, 3), dt, dx, G, 1 - sweep)
    assert np.abs(other - out).max() > 1e-9


def test_decomposition_invariance_and_group_layout():
    """Per-group results (N = 8, ghost shells cut from the padded box) equal the whole-box result bit for bit."""
    n = 16
    U = smooth_box(n, 6)
    dt, dx = 0.01, 1.0 / n
    whole = R.step_box(wl.pad_box(U, ("periodic",) * 3, 3), dt, dx, G, 0)
    grp = wl.cut_groups(U, ("periodic",) * 3, N=8, ghost=3, dtype=np.float64)
    out, _ = R.step_groups(grp, 8, dt, dx, G, 0)
    assert np.array_equal(wl.assemble_box(out, (n, n, n), N=8), whole)


def test_conservation_in_a_periodic_box():
    n = 16
    U = smooth_box(n, 7)
    V = U.copy()
    for s in range(6):
        V = R.step_box(wl.pad_box(V, ("periodic",) * 3, 3), 0.004, 1.0 / n, G, s % 2)
    for q in range(5):
        assert abs(V[q].sum() - U[q].sum()) <= 1e-12 * np.abs(U[q]).sum(), q


def test_axis_permutation_maps_sweep_xyz_on_zyx():
    """Relabelling the axes x <-> z (array transpose + momentum swap) turns the x,y,z step into the z,y,x step."""
    n = 8
    U = smooth_box(n, 8)
    dt, dx = 0.005, 1.0 / n
    a = R.step_box(wl.pad_box(U, ("periodic",) * 3, 3), dt, dx, G, 0)
    Ut = U.transpose(0, 3, 2, 1)[[0, 3, 2, 1, 4]]
    b = R.step_box(wl.pad_box(np.ascontiguousarray(Ut), ("periodic",) * 3, 3), dt, dx, G, 1)
    back = b.transpose(0, 3, 2, 1)[[0, 3, 2, 1, 4]]
    assert np.abs(back - a).max() <= 1e-13 * np.abs(a).max()


def _sod_line(nx, steps, cfl=0.5):
    """Sod tube along x, advanced with the 1-D sweep only (y, z uniform: the other sweeps are identities up to
    round-off, checked separately); outflow ends; dt = C dx / max(|v| + c_s)."""
    x = (np.arange(nx) + 0.5) / nx
    u = np.array([cons(1, 0, 0, 0, 1) if xx < 0.5 else cons(0.125, 0, 0, 0, 0.1) for xx in x])
    t = 0.0
    for _ in range(steps):
        rho = u[:, 0]; v = u[:, 1] / rho
        P = (G - 1) * (u[:, 4] - 0.5 * rho * v * v)
        dt = cfl / nx / np.max(np.abs(v) + np.sqrt(G * P / rho))
        padded = np.concatenate([np.repeat(u[:1], 3, 0), u, np.repeat(u[-1:], 3, 0)])
        u = R.sweep_line(padded, 0, dt, 1.0 / nx, G)[3:-3]
        t += dt
    return u, t


def test_sod_tube_against_the_exact_riemann_solution():
    errs = {}
    for nx in (256, 512):
        u, t = _sod_line(nx, nx // 4)
        x = (np.arange(nx) + 0.5) / nx
        rho_e, u_e, p_e = er.sample(G, (1, 0, 1), (0.125, 0, 0.1), (x - 0.5) / t)
        errs[nx] = float(np.mean(np.abs(u[:, 0] - rho_e)))
        assert u[:, 0].max() <= 1.0 + 1e-12 and u[:, 0].min() >= 0.125 - 1e-12     # no new extrema
        tv = np.abs(np.diff(u[:, 0])).sum()
        assert tv <= 0.875 * 1.05                  # no oscillations: the variation stays within 5 % of the initial jump (a system,
                                                   # not a scalar law: the strict TVD bound holds per relaxed wave, not for rho)
        if nx == 512:
            xi = (x - 0.5) / t
            starR = (xi > 0.8411948522 + 0.3) & (xi < 1.844473367 - 0.25)           # SURVEY.md App. A constants
            rho = u[:, 0]; v = u[:, 1] / rho; P = (G - 1) * (u[:, 4] - 0.5 * rho * v * v)
            assert starR.sum() >= 8
            assert np.allclose(rho[starR], 0.2298057493, rtol=2e-2) and np.allclose(P[starR], 0.2939451877, rtol=2e-2)
            assert np.allclose(v[starR], 0.8411948522, rtol=2e-2)
    assert 1.4 <= errs[256] / errs[512] <= 2.6, errs        # about first order for a solution with discontinuities


def test_second_order_convergence_on_a_smooth_entropy_wave():
    """rho = 1 + 0.2 sin(2 pi x), uniform v and P, periodic: an exact solution is the translated profile."""
    errs = {}
    for nx in (32, 64, 128):
        x = (np.arange(nx) + 0.5) / nx
        v0, P0 = 1.0, 1.0
        u = np.array([cons(1 + 0.2 * np.sin(2 * np.pi * xx), v0, 0, 0, P0) for xx in x])
        cmax = v0 + np.sqrt(G * P0 / 0.8)
        steps = nx // 2
        dt = 0.4 / nx / cmax
        for _ in range(steps):
            padded = np.concatenate([u[-3:], u, u[:3]])
            u = R.sweep_line(padded, 0, dt, 1.0 / nx, G)[3:-3]
        exact = 1 + 0.2 * np.sin(2 * np.pi * (x - v0 * dt * steps))
        errs[nx] = float(np.mean(np.abs(u[:, 0] - exact)))
    assert errs[32] / errs[64] >= 3.0 and errs[64] / errs[128] >= 3.0, errs      # limiter clipping keeps it a little under 4


def test_one_dimensional_data_stay_one_dimensional_in_3d():
    """x-dependent data in a 3-D box: the y and z sweeps are exact identities (uniform lines), transverse momenta stay
    exactly zero, and every (y, z) column equals the 1-D sweep."""
    nx = 32
    x = (np.arange(nx) + 0.5) / nx
    line = np.array([cons(1 + 0.3 * np.sin(2 * np.pi * xx), 0.4, 0, 0, 1 + 0.2 * np.cos(2 * np.pi * xx)) for xx in x])
    box = np.broadcast_to(line.T[:, None, None, :], (5, 8, 8, nx)).copy()
    dt, dx = 0.004, 1.0 / nx
    for sweep in (0, 1):
        out = R.step_box(wl.pad_box(box, ("periodic",) * 3, 3), dt, dx, G, sweep)
        ref = R.sweep_line(np.concatenate([line[-3:], line, line[:3]]), 0, dt, dx, G)[3:-3]
        assert np.array_equal(out[2], np.zeros_like(out[2])) and np.array_equal(out[3], np.zeros_like(out[3]))
        assert np.array_equal(out[:, 2, 5, :], ref.T) and np.array_equal(out[:, 7, 0, :], ref.T)


def test_flop_tally_matches_a_hand_count_of_the_oracle_text():
    """The roofline numerator of bench.py's relaxing-TVD leg (RTVD_FLOPS_PER_CELL) is the oracle text run with a counting
    scalar. Pin: the count typed out here by hand from the text of sweep_line, per line of L cells, convention of
    oracle/counting_real.hpp (add = sub = mul = div = sqrt = 1; abs, negate, compare, select = 0):
      flux_and_speed 21 per cell (v 1; ke 7; P 3; F 6; c 4) + the split fluxes 2 x 3 x 5 = 30   -> 51 per cell
      half step: 51 L + 5 (L-1) first-order face fluxes + 20 (L-2) for the half-step state
      full step: 51 (L-2) + 95 (L-5) limited face fluxes (19 per variable) + 15 (L-6) update; 1 for lambda = dt/dx
    over the 22^2 + 22*16 + 16^2 = 1092 lines a 16^3 group's three sweeps touch (RT5: the range shrinks after a sweep).
    Opposite-sign differences skip the 4 operations of the van Leer quotient, so the tally may sit slightly below."""
    import bench
    L, N = 22, 16
    per_line = 51 * L + 5 * (L - 1) + 20 * (L - 2) + 51 * (L - 2) + 95 * (L - 5) + 15 * (L - 6) + 1
    lines = L * L + L * N + N * N
    hand = per_line * lines / float(N ** 3)
    assert per_line == 4503 and lines == 1092 and abs(hand - 1200.5) < 0.05
    z, y, x = np.meshgrid(*(np.arange(L, dtype=np.float64),) * 3, indexing="ij")
    ramp = 1.0 + 0.01 * (x + 2 * y + 3 * z)          # monotone along every axis: (almost) every limiter active
    U = wl.prim_box_to_cons(ramp, 0.1 * ramp, -0.2 * ramp, 0.3 * ramp, 2.0 * ramp)
    for sweep in (0, 1):
        c = R.count_flops(U, N, 1e-3, 1 / 16, G, sweep)
        assert c["sqrt"] == lines * (2 * L - 2) and c["minmax"] == 0
        assert 0.999 * hand <= c["per_cell"] <= hand, (c, hand)
        assert abs(bench.RTVD_FLOPS_PER_CELL - c["per_cell"]) <= 1.0, (bench.RTVD_FLOPS_PER_CELL, c["per_cell"])
