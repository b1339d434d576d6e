"""Pins of the robustness variants of the oracle: MC limiter, Harten-Hyman
entropy fix, HLLE fallback, mid-plane fluxes. Closed forms, exact Riemann solutions and invariants; CPU only."""
import math

import numpy as np
import pytest

import exact_riemann as er
from harness import workloads as wl
from oracle import mhm_oracle as O

G53 = 5.0 / 3.0


def cons(rho, vx, vy, vz, P, g):
    return np.array([rho, rho * vx, rho * vy, rho * vz, P / (g - 1) + 0.5 * rho * (vx * vx + vy * vy + vz * vz)])


def euler_flux(rho, vx, vy, vz, P, d, g):
    v = (vx, vy, vz)
    E = P / (g - 1) + 0.5 * rho * (vx * vx + vy * vy + vz * vz)
    F = np.array([rho * v[d], rho * vx * v[d], rho * vy * v[d], rho * vz * v[d], (E + P) * v[d]])
    F[1 + d] += P
    return F


# ------------------------------------------------------------------ MC limiter

def test_mc_limiter_hand_values_and_tvd_bound():
    assert O.limited_slope(1.0, 3.0, 2) == 2.0          # min(2, 6, 2)
    assert O.limited_slope(1.0, 1.2, 2) == pytest.approx(1.1, abs=1e-15)   # the central difference wins
    assert O.limited_slope(3.0, 0.5, 2) == 1.0          # min(6, 1, 1.75)
    assert O.limited_slope(-1.0, -3.0, 2) == -2.0
    assert O.limited_slope(1.0, -1.0, 2) == 0.0 and O.limited_slope(0.0, 2.0, 2) == 0.0
    rng = np.random.default_rng(1)
    for a, b in rng.normal(0, 1, (500, 2)):
        s = O.limited_slope(a, b, 2)
        if a * b <= 0:
            assert s == 0.0
        else:
            assert abs(s) <= 2 * min(abs(a), abs(b)) * (1 + 1e-15) and s * a > 0
            assert abs(s) >= min(abs(a), abs(b)) * (1 - 1e-15)      # MC is never more diffusive than MinMod
    for k in (0.3, -2.0):                                            # a linear field keeps its slope exactly
        assert O.limited_slope(k, k, 2) == k


def test_mc_step_is_second_order_and_sharper_than_minmod():
    """Smooth entropy wave, periodic, one period fraction: L1 error falls by > 3.3 per halving with MC, and is
    below MinMod's at the same resolution."""
    errs = {0: {}, 2: {}}
    for lim in (0, 2):
        for n in (16, 32):
            x = (np.arange(n) + 0.5) / n
            rho = 1 + 0.2 * np.sin(2 * np.pi * x)
            one = np.ones((16, 16, n))
            U = wl.prim_box_to_cons(rho[None, None, :] * one, one, 0 * one, 0 * one, one)
            dx = 1.0 / n
            dt = 0.3 * dx / (1 + 3 * math.sqrt(G53 / 0.8))
            steps = n // 2
            for _ in range(steps):
                r, _m = O.step_groups_ex(wl.cut_groups(U, ("periodic",) * 3, dtype=np.float64), 16, 2, dt, dx, G53, lim)
                U = wl.assemble_box(r.U_out, (16, 16, n))
            exact = 1 + 0.2 * np.sin(2 * np.pi * (x - dt * steps))
            errs[lim][n] = float(np.mean(np.abs(U[0, 3, 5, :] - exact)))
    assert errs[2][16] / errs[2][32] >= 3.3, errs
    assert errs[2][32] < errs[0][32], errs


# ------------------------------------------------------------------ entropy fix

def _transonic_pair(g=1.4):
    # Toro's test 1: left (1, 0.75, 1), right (0.125, 0, 0.1): the left rarefaction contains a sonic point
    return (1.0, 0.75, 1.0), (0.125, 0.0, 0.1)


def test_entropy_fix_moves_the_transonic_flux_towards_the_exact_godunov_flux():
    """Two states taken from ONE rarefaction fan on either side of its sonic point (the exact solution of Toro's test 1
    at xi = -0.2 and +0.2): the exact Godunov flux between them is the flux at the sonic point. Plain Roe, whose
    averaged acoustic speed nearly vanishes there, returns about the mean of the two fluxes (the expansion shock); the
    fix brings the flux several times closer (for Burgers' equation it is exact)."""
    g = 1.4
    L, Rr = _transonic_pair()
    rho, u, p = er.sample(g, L, Rr, np.array([-0.2, 0.0, 0.2]))
    assert abs(u[1] - math.sqrt(g * p[1] / rho[1])) < 1e-8               # xi = 0 is the sonic point of the fan
    UL, UR = cons(rho[0], u[0], 0, 0, p[0], g), cons(rho[2], u[2], 0, 0, p[2], g)
    F_exact = euler_flux(rho[1], u[1], 0, 0, p[1], 0, g)
    F_plain = O.roe_flux(UL, UR, g, 0)
    F_fix, used = O.roe_flux_ex(UL, UR, g, 0, O.ENTROPY_FIX)
    assert not used
    e_plain, e_fix = np.abs(F_plain - F_exact).max(), np.abs(F_fix - F_exact).max()
    assert e_fix < 0.25 * e_plain, (e_plain, e_fix)


def test_entropy_fix_is_inactive_away_from_transonic_expansions():
    rng = np.random.default_rng(2)
    g = G53
    n_same = 0
    for _ in range(300):
        rho, P = rng.uniform(0.5, 2, 2), rng.uniform(0.5, 2, 2)
        u0 = rng.choice([-4.0, 4.0])                                     # supersonic on both sides: no sonic point
        UL = cons(rho[0], u0 + rng.normal(0, 0.1), rng.normal(), rng.normal(), P[0], g)
        UR = cons(rho[1], u0 + rng.normal(0, 0.1), rng.normal(), rng.normal(), P[1], g)
        for d in range(3):
            rot = lambda U: U[[0, 1 + (0 - d) % 3, 1 + (1 - d) % 3, 1 + (2 - d) % 3, 4]]
            a, b = O.roe_flux(rot(UL), rot(UR), g, d), O.roe_flux_ex(rot(UL), rot(UR), g, d, O.ENTROPY_FIX)[0]
            n_same += int(np.array_equal(a, b))
    assert n_same == 900
    U = cons(1.3, 0.37, -0.61, 0.23, 0.9, g)                              # consistency stays bit-exact
    for d in range(3):
        assert np.array_equal(O.roe_flux_ex(U, U, g, d, 3)[0], O.phys_flux(U, g, d))


def _tube(states, g, nx, steps_t, limiter, flags, cfl=0.4):
    """1-D Riemann problem along x in a 16 x 16 x nx box, outflow ends; returns (rho(x), t) or None if the run died."""
    L, Rr = states
    x = (np.arange(nx) + 0.5) / nx
    left = (x < 0.5)[None, None, :] * np.ones((16, 16, nx), dtype=bool)
    pick = lambda a, b: np.where(left, a, b)
    z = np.zeros((16, 16, nx))
    U = wl.prim_box_to_cons(pick(L[0], Rr[0]) + z, pick(L[1], Rr[1]) + z, z, z, pick(L[2], Rr[2]) + z, g)
    bc = ("outflow", "periodic", "periodic")
    t = 0.0
    while t < steps_t:
        vmax = wl.max_signal_speed(U, g)
        if not np.isfinite(vmax):
            return None, t
        dt = min(cfl / nx / vmax, steps_t - t)
        r, _m = O.step_groups_ex(wl.cut_groups(U, bc, dtype=np.float64), 16, 2, dt, 1.0 / nx, g, limiter, flags)
        U = wl.assemble_box(r.U_out, (16, 16, nx))
        if not np.isfinite(U).all() or U[0].min() <= 0:
            return None, t
        t += dt
    return U, t


def test_entropy_fix_removes_the_expansion_shock_of_toro_test_1():
    """The glitch of plain Roe at the sonic point: a density jump across one face inside the smooth rarefaction. With
    the fix the largest cell-to-cell jump inside the fan is close to the exact profile's slope times dx."""
    g, nx, T = 1.4, 128, 0.15
    out = {}
    for flags in (0, O.ENTROPY_FIX):
        U, t = _tube(_transonic_pair(), g, nx, T, 0, flags)
        assert U is not None
        x = (np.arange(nx) + 0.5) / nx
        xi = (x - 0.5) / t
        rho_e, u_e, p_e = er.sample(g, *_transonic_pair(), xi)
        rho = U[0, 3, 5, :]
        fan = (xi > -0.35) & (xi < 0.25)                                  # around the sonic point xi = 0
        out[flags] = (float(np.mean(np.abs(rho - rho_e))), float(np.abs(np.diff(rho[fan])).max()),
                      float(np.abs(np.diff(rho_e[fan])).max()))
    l1_plain, jump_plain, slope = out[0]
    l1_fix, jump_fix, _ = out[O.ENTROPY_FIX]
    assert jump_fix <= 1.6 * slope, out                                   # smooth through the sonic point
    assert jump_plain >= 1.3 * jump_fix, out                              # plain Roe shows the glitch
    assert l1_fix <= l1_plain * 1.001, out


# ------------------------------------------------------------------ HLLE fallback

def test_hlle_fallback_formula_detection_and_identity_elsewhere():
    g = 1.4
    UL, UR = cons(1, -2, 0, 0, 0.4, g), cons(1, 2, 0, 0, 0.4, g)          # Toro's test 2: strong double rarefaction
    F, used = O.roe_flux_ex(UL, UR, g, 0, O.HLLE_FALLBACK)
    assert used
    aL = aR = math.sqrt(g * 0.4 / 1.0)
    bm, bp = min(-2 - aL, 0.0), max(2 + aR, 0.0)                          # Roe averages: u~ = 0, so the outer speeds win
    FL, FR = euler_flux(1, -2, 0, 0, 0.4, 0, g), euler_flux(1, 2, 0, 0, 0.4, 0, g)
    want = (bp * FL - bm * FR + bp * bm * (UR - UL)) / (bp - bm)
    assert np.allclose(F, want, rtol=1e-14, atol=1e-14)
    # the plain intermediate state is indeed non-physical: rho* = rho_L + alpha_1 < 0
    al, lam, K = O.roe_decompose(UL, UR, g, 0)
    assert 1.0 + al[0] < 0
    # moderate jumps have physical intermediate states: the flag changes nothing, bit for bit
    rng = np.random.default_rng(3)
    for _ in range(300):
        A = cons(rng.uniform(0.8, 1.25), *rng.normal(0, 0.2, 3), rng.uniform(0.8, 1.25), g)
        B = cons(rng.uniform(0.8, 1.25), *rng.normal(0, 0.2, 3), rng.uniform(0.8, 1.25), g)
        for d in range(3):
            Fh, used = O.roe_flux_ex(A, B, g, d, O.HLLE_FALLBACK)
            assert not used and np.array_equal(Fh, O.roe_flux(A, B, g, d))


def test_hlle_fallback_keeps_the_double_rarefaction_positive_where_plain_roe_fails():
    g, nx, T = 1.4, 128, 0.06
    states = ((1.0, -2.0, 0.4), (1.0, 2.0, 0.4))
    U_plain, t_plain = _tube(states, g, nx, T, 0, 0)
    U_fb, t = _tube(states, g, nx, T, 0, O.HLLE_FALLBACK)
    assert U_fb is not None and abs(t - T) < 1e-12
    rho = U_fb[0]
    P = (g - 1) * (U_fb[4] - 0.5 * (U_fb[1] ** 2 + U_fb[2] ** 2 + U_fb[3] ** 2) / rho)
    assert rho.min() > 0 and P.min() > 0
    if U_plain is not None:                                                # plain Roe either dies or leaves P <= 0 behind
        Pp = (g - 1) * (U_plain[4] - 0.5 * (U_plain[1] ** 2 + U_plain[2] ** 2 + U_plain[3] ** 2) / U_plain[0])
        assert Pp.min() <= 0
    x = (np.arange(nx) + 0.5) / nx
    rho_e, u_e, p_e = er.sample(g, *states, (x - 0.5) / t)
    assert float(np.mean(np.abs(rho[3, 5, :] - rho_e))) < 0.05             # and it is the right solution


# ------------------------------------------------------------------ mid-plane fluxes

@pytest.mark.parametrize("limiter", [0, 2])
def test_midplane_fluxes_balance_each_half_of_a_group(limiter):
    """A group of 2 x 2 x 2 patches: for each axis, the lower half of the group balances with the outer-face fluxes
    of that half and the mid-plane flux (reading R12b): sum(U_out - U_in) = -lambda * (net outflow of the half)."""
    g = wl.random_groups(3, seed=55, dtype=np.float64)
    dt, dx = 2e-3, 1.0 / 16
    lam = dt / dx
    r, mf = O.step_groups_ex(g, 16, 2, dt, dx, G53, limiter, 0, want_midflux=True)
    assert mf.shape == (3, 3, 5, 16, 16)
    dU = r.U_out - g[:, :, 2:-2, 2:-2, 2:-2]
    bf = r.bflux                                                            # [G][6][5][N][N]
    H = slice(0, 8)
    for n in range(3):
        # x half (i < 8): x faces [k][j], y faces [k][i], z faces [j][i]
        lhs = dU[n][:, :, :, H].sum(axis=(1, 2, 3))
        net = (mf[n, 0].sum(axis=(1, 2)) - bf[n, 0].sum(axis=(1, 2))) + \
              (bf[n, 3][:, :, H].sum(axis=(1, 2)) - bf[n, 2][:, :, H].sum(axis=(1, 2))) + \
              (bf[n, 5][:, :, H].sum(axis=(1, 2)) - bf[n, 4][:, :, H].sum(axis=(1, 2)))
        assert np.allclose(lhs, -lam * net, rtol=1e-11, atol=1e-11)
        # y half (j < 8)
        lhs = dU[n][:, :, H, :].sum(axis=(1, 2, 3))
        net = (mf[n, 1].sum(axis=(1, 2)) - bf[n, 2].sum(axis=(1, 2))) + \
              (bf[n, 1][:, :, H].sum(axis=(1, 2)) - bf[n, 0][:, :, H].sum(axis=(1, 2))) + \
              (bf[n, 5][:, H, :].sum(axis=(1, 2)) - bf[n, 4][:, H, :].sum(axis=(1, 2)))
        assert np.allclose(lhs, -lam * net, rtol=1e-11, atol=1e-11)
        # z half (k < 8)
        lhs = dU[n][:, H, :, :].sum(axis=(1, 2, 3))
        net = (mf[n, 2].sum(axis=(1, 2)) - bf[n, 4].sum(axis=(1, 2))) + \
              (bf[n, 1][:, H, :].sum(axis=(1, 2)) - bf[n, 0][:, H, :].sum(axis=(1, 2))) + \
              (bf[n, 3][:, H, :].sum(axis=(1, 2)) - bf[n, 2][:, H, :].sum(axis=(1, 2)))
        assert np.allclose(lhs, -lam * net, rtol=1e-11, atol=1e-11)
    # a hot cell next to the x mid-plane pins the in-face (k, j) order
    U = wl.prim_box_to_cons(*(np.full((16, 16, 16), v) for v in (1.0, 0.0, 0.0, 0.0, 1.0)))
    U[4, 5, 11, 7] *= 3.0                                                   # cell (i = 7, j = 11, k = 5)
    r2, mf2 = O.step_groups_ex(wl.cut_groups(U, ("periodic",) * 3, dtype=np.float64), 16, 2, dt, dx, G53, 0, 0, True)
    dev = np.abs(mf2[0, 0, 1] - mf2[0, 0, 1, 0, 0])                         # x-momentum flux on the x mid-plane, [k][j]
    assert np.unravel_index(dev.argmax(), dev.shape) == (5, 11)
    # default arguments reproduce the plain step bit for bit
    r0 = O.step_groups(g, 16, 2, dt, dx, G53, 0)
    r1, _ = O.step_groups_ex(g, 16, 2, dt, dx, G53, 0)
    assert np.array_equal(r0.U_out, r1.U_out) and np.array_equal(r0.bflux, r1.bflux)


def test_hlle_face_map_marks_exactly_the_faces_whose_flux_changed():
    """Pin of the diagnostic map step_groups_ex(want_hlle=True) returns (the parity harness' face-level accounting of the
    HLLE switch rests on its layout [g][axis][k][j][i], face on the lower side of cell (i, j, k)): no face is marked
    without the flag; with it, a cell none of whose six faces is marked is updated bit for bit as by plain Roe, a cell
    next to a marked face generally is not; and the marked outer faces are exactly those whose boundary flux changed."""
    import numpy as np
    from harness import workloads as wl
    g = wl.random_groups(2, seed=302, mach=2.0, contrast=0.8)
    dt, dx, gam = 5e-4, 1 / 16, 5.0 / 3.0
    r0, _ = O.step_groups_ex(g, 16, 2, dt, dx, gam, 1, 0, want_hlle=True)
    r2, _ = O.step_groups_ex(g, 16, 2, dt, dx, gam, 1, 2, want_hlle=True)
    assert r0.hlle.sum() == 0 and r2.hlle.sum() > 1000
    h = r2.hlle != 0
    for absent in (h[:, 0, 16], h[:, 0, :, 16], h[:, 1, 16], h[:, 1, :, :, 16], h[:, 2, :, 16], h[:, 2, :, :, 16]):
        assert not absent.any()                                                    # faces that do not exist stay 0
    hx, hy, hz = h[:, 0, :16, :16, :], h[:, 1, :16, :, :16], h[:, 2, :, :16, :16]
    touched = (hx[..., :16] | hx[..., 1:]) | (hy[:, :, :16, :] | hy[:, :, 1:, :]) | (hz[:, :16] | hz[:, 1:])
    same = np.all(r0.U_out == r2.U_out, axis=1)
    assert same[~touched].all()                                                    # untouched cells: plain Roe bits
    assert (~same[touched]).mean() > 0.9                                           # touched cells: the flux changed
    outer = [hx[..., 0], hx[..., 16], hy[:, :, 0, :], hy[:, :, 16, :], hz[:, 0], hz[:, 16]]
    for f in range(6):
        changed = np.any(r0.bflux[:, f] != r2.bflux[:, f], axis=1)
        assert not changed[~outer[f]].any() and changed[outer[f]].mean() > 0.9
