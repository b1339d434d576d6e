"""Second, deliberately different transcriptions of the method, written from the same passages
(SURVEY.md §8(c) O1–O7) but sharing no loops, helpers or formula variants with oracle/:

* step_group_naive — whole-array numpy slicing on one patch group, Roe flux in the Roe–Pike primitive-jump
  form (alpha_1,5 = (dp -+ rho~ a~ du)/(2 a~^2), alpha_2 = drho - dp/a~^2, alpha_3,4 = rho~ dv, rho~ dw,
  rho~ = sqrt(rhoL rhoR)), the oracle uses the conserved-jump form, so agreement also checks the identity
  (pin P16).
* mhm_1d — a 1-D MUSCL-Hancock + 3-wave Roe solver in the textbook form (Toro 2009 §14.4 / §11.2), for the
  1-D reduction pin P14.
Both are TEST code. Neither is used by the product or by the oracle."""
import numpy as np


def _sl(a, axis, lo, hi):
    idx = [slice(None)] * a.ndim
    idx[axis] = slice(lo, hi if hi != 0 else None)
    return a[tuple(idx)]


def _slope(dL, dR, limiter):
    same = ((dL > 0) & (dR > 0)) | ((dL < 0) & (dR < 0))
    if limiter == 0:
        s = np.sign(dL) * np.minimum(np.abs(dL), np.abs(dR))
    else:
        with np.errstate(divide="ignore", invalid="ignore"):
            s = 2.0 * dL * dR / (dL + dR)
    return np.where(same, s, 0.0)


def _cons(W, g):
    U = np.empty_like(W)
    U[0] = W[0]
    U[1:4] = W[0] * W[1:4]
    U[4] = W[4] / (g - 1.0) + 0.5 * W[0] * (W[1] ** 2 + W[2] ** 2 + W[3] ** 2)
    return U


def _prim(U, g):
    W = np.empty_like(U)
    W[0] = U[0]
    W[1:4] = U[1:4] / U[0]
    W[4] = (g - 1.0) * (U[4] - 0.5 * (U[1] * W[1] + U[2] * W[2] + U[3] * W[3]))
    return W


def _flux(U, W, comp):
    F = np.empty_like(U)
    vn = W[1 + comp]
    F[0] = U[1 + comp]
    for q in (1, 2, 3):
        F[q] = U[q] * vn
    F[1 + comp] = F[1 + comp] + W[4]
    F[4] = (U[4] + W[4]) * vn
    return F


def _roe_pike(UL, UR, g, comp):
    n, t1, t2 = 1 + comp, 1 + (comp + 1) % 3, 1 + (comp + 2) % 3
    WL, WR = _prim(UL, g), _prim(UR, g)
    HL, HR = (UL[4] + WL[4]) / UL[0], (UR[4] + WR[4]) / UR[0]
    sl, sr = np.sqrt(UL[0]), np.sqrt(UR[0])
    avg = lambda a, b: (sl * a + sr * b) / (sl + sr)
    u, v, w, H = avg(WL[n], WR[n]), avg(WL[t1], WR[t1]), avg(WL[t2], WR[t2]), avg(HL, HR)
    q2 = u * u + v * v + w * w
    a2 = (g - 1.0) * (H - 0.5 * q2)
    a = np.sqrt(a2)
    rt = sl * sr
    dr, du, dv, dw, dp = WR[0] - WL[0], WR[n] - WL[n], WR[t1] - WL[t1], WR[t2] - WL[t2], WR[4] - WL[4]
    al = [(dp - rt * a * du) / (2 * a2), dr - dp / a2, rt * dv, rt * dw, (dp + rt * a * du) / (2 * a2)]
    lam = [np.abs(u - a), np.abs(u), np.abs(u), np.abs(u), np.abs(u + a)]
    one, zero = np.ones_like(u), np.zeros_like(u)
    K = [[one, u - a, v, w, H - u * a], [one, u, v, w, 0.5 * q2], [zero, zero, one, zero, v],
         [zero, zero, zero, one, w], [one, u + a, v, w, H + u * a]]
    FL, FR = _flux(UL, WL, comp), _flux(UR, WR, comp)
    order = [0, n, t1, t2, 4]
    F = np.empty_like(UL)
    for c in range(5):
        diss = sum(al[i] * lam[i] * K[i][c] for i in range(5))
        F[order[c]] = 0.5 * (FL[order[c]] + FR[order[c]]) - 0.5 * diss
    return F


def step_group_naive(U_in, N, ghost, dt, dx, gamma, limiter):
    """One step on one group U_in [5][S][S][S] (fp64). Returns (U_out [5][N][N][N], bflux [6][5][N][N],
    guard [N+2]^3 bool)."""
    g = gamma
    U = np.asarray(U_in, dtype=np.float64)
    o = ghost - 2
    if o:
        U = U[:, o:-o, o:-o, o:-o]
    with np.errstate(all="ignore"):
        W = _prim(U, g)                       # 20^3
        core = W[:, 1:-1, 1:-1, 1:-1]         # 18^3: cells -1..N
        lam = dt / dx
        Uf = {}
        dF = 0.0
        for comp, axis in ((0, 3), (1, 2), (2, 1)):
            other = [ax for ax in (1, 2, 3) if ax != axis]
            Wm1 = _sl(_sl(_sl(W, axis, 0, -2), other[0], 1, -1), other[1], 1, -1)
            Wp1 = _sl(_sl(_sl(W, axis, 2, 0), other[0], 1, -1), other[1], 1, -1)
            s = _slope(core - Wm1, Wp1 - core, limiter)
            Wminus, Wplus = core - 0.5 * s, core + 0.5 * s
            Uminus, Uplus = _cons(Wminus, g), _cons(Wplus, g)
            Uf[comp] = (Uminus, Uplus)
            dF = dF + (_flux(Uplus, Wplus, comp) - _flux(Uminus, Wminus, comp))
        dU = -0.5 * lam * dF
        ok = np.ones(core.shape[1:], dtype=bool)
        for comp in range(3):
            for Us in Uf[comp]:
                Ub = Us + dU
                ok &= (Ub[0] > 0) & (2 * Ub[0] * Ub[4] > Ub[1] ** 2 + Ub[2] ** 2 + Ub[3] ** 2)
        Ucell = U[:, 1:-1, 1:-1, 1:-1]
        Ubar = {c: tuple(np.where(ok, Us + dU, Ucell) for Us in Uf[c]) for c in range(3)}
        out = U[:, 2:-2, 2:-2, 2:-2].copy()
        bflux = np.empty((6, 5, N, N))
        tot = 0.0
        for comp, axis in ((0, 3), (1, 2), (2, 1)):
            other = [ax for ax in (1, 2, 3) if ax != axis]
            inner = lambda A: _sl(_sl(A, other[0], 1, -1), other[1], 1, -1)
            UL = _sl(inner(Ubar[comp][1]), axis, 0, -1)   # '+' state of cells -1..N-1
            UR = _sl(inner(Ubar[comp][0]), axis, 1, 0)    # '-' state of cells 0..N
            F = _roe_pike(UL, UR, g, comp)                # N+1 faces along axis
            tot = tot + (_sl(F, axis, 1, 0) - _sl(F, axis, 0, -1))
            bflux[2 * comp] = np.take(F, 0, axis=axis)
            bflux[2 * comp + 1] = np.take(F, N, axis=axis)
        out = out - lam * tot
    return out, bflux, ~ok


# ------------------------------------------------------------------------------------------------------
# 1-D MUSCL-Hancock with a 3-wave Roe solver (textbook form), periodic or outflow ends.


def _prim1(U, g):
    r, m, E = U
    u = m / r
    return r, u, (g - 1.0) * (E - 0.5 * m * u)


def _flux1(r, u, p, g):
    E = p / (g - 1.0) + 0.5 * r * u * u
    return np.array([r * u, r * u * u + p, (E + p) * u])


def _roe1(UL, UR, g):
    rl, ul, pl = _prim1(UL, g)
    rr, ur, pr = _prim1(UR, g)
    hl, hr = (UL[2] + pl) / rl, (UR[2] + pr) / rr
    sl, sr = np.sqrt(rl), np.sqrt(rr)
    u = (sl * ul + sr * ur) / (sl + sr)
    H = (sl * hl + sr * hr) / (sl + sr)
    a = np.sqrt((g - 1.0) * (H - 0.5 * u * u))
    d1, d2, d3 = UR[0] - UL[0], UR[1] - UL[1], UR[2] - UL[2]
    a2 = (g - 1.0) / (a * a) * (d1 * (H - u * u) + u * d2 - d3)
    a1 = (d1 * (u + a) - d2 - a * a2) / (2.0 * a)
    a3 = d1 - (a1 + a2)
    K1, K2, K3 = np.array([np.ones_like(u), u - a, H - u * a]), np.array([np.ones_like(u), u, 0.5 * u * u]), \
        np.array([np.ones_like(u), u + a, H + u * a])
    diss = a1 * np.abs(u - a) * K1 + a2 * np.abs(u) * K2 + a3 * np.abs(u + a) * K3
    return 0.5 * (_flux1(rl, ul, pl, g) + _flux1(rr, ur, pr, g)) - 0.5 * diss


def mhm_1d(U, dt, dx, g, limiter, bc):
    """U [3][n] (rho, m, E) -> one step; bc 'periodic' or 'outflow'."""
    n = U.shape[1]
    Up = np.pad(U, ((0, 0), (2, 2)), mode="wrap" if bc == "periodic" else "edge")
    r, u, p = _prim1(Up, g)
    W = np.array([r, u, p])
    c = W[:, 1:-1]
    s = _slope(c - W[:, :-2], W[:, 2:] - c, limiter)
    Wl, Wr = c - 0.5 * s, c + 0.5 * s
    cons = lambda w: np.array([w[0], w[0] * w[1], w[2] / (g - 1.0) + 0.5 * w[0] * w[1] ** 2])
    Ul, Ur = cons(Wl), cons(Wr)
    dU = -0.5 * dt / dx * (_flux1(*Wr, g) - _flux1(*Wl, g))
    Ul, Ur = Ul + dU, Ur + dU
    F = _roe1(Ur[:, :-1], Ul[:, 1:], g)  # n+1 faces
    return U - dt / dx * (F[:, 1:] - F[:, :-1])
