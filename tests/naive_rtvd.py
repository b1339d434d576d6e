"""A second, independent transcription of the relaxing-TVD step (Trac & Pen 2003), used to pin oracle/rtvd_oracle.hpp
(brute-force pin): WHOLE periodic arrays moved with numpy circular shifts — no ghost cells, no lines, no index
ranges — so that an indexing or ghost-accounting mistake in the oracle's loops cannot be shared. Pure numpy, fp64."""
import numpy as np


def _flux_speed(u, d, g):
    """u: [5, ...]; returns (F_d(u), c) with c = |v_d| + c_s."""
    rho = u[0]
    v = u[1 + d] / rho
    P = (g - 1.0) * (u[4] - 0.5 * (u[1] ** 2 + u[2] ** 2 + u[3] ** 2) / rho)
    F = np.stack([u[1 + d], u[1] * v, u[2] * v, u[3] * v, (u[4] + P) * v])
    F[1 + d] = F[1 + d] + P
    return F, np.abs(v) + np.sqrt(g * np.maximum(P, 0.0) / rho)


def _vanleer(a, b):
    ok = ((a > 0) & (b > 0)) | ((a < 0) & (b < 0))
    den = np.where(ok, a + b, 1.0)
    return np.where(ok, 2.0 * a * b / den, 0.0)


def sweep_periodic(u, d, dt, dx, g):
    """One sweep along axis d of a periodic box u [5][nz][ny][nx] (array axis of d: 3 - d)."""
    ax = 3 - d
    sh = lambda a, k: np.roll(a, -k, axis=ax)        # sh(a, 1)[j] = a[j+1]
    lam = dt / dx
    F, c = _flux_speed(u, d, g)
    fr = 0.5 * (c * u + F)
    fl = 0.5 * (c * u - F)
    fu = fr - sh(fl, 1)                              # face j+1/2
    u1 = u - 0.5 * lam * (fu - sh(fu, -1))
    F, c = _flux_speed(u1, d, g)
    fr = 0.5 * (c * u1 + F)
    fl = 0.5 * (c * u1 - F)
    FR = fr + _vanleer(0.5 * (fr - sh(fr, -1)), 0.5 * (sh(fr, 1) - fr))
    FL = sh(fl, 1) + _vanleer(0.5 * (fl - sh(fl, 1)), 0.5 * (sh(fl, 1) - sh(fl, 2)))
    fu = FR - FL
    return u - lam * (fu - sh(fu, -1))


def step_periodic(u, dt, dx, g, sweep):
    order = (0, 1, 2) if sweep == 0 else (2, 1, 0)
    for d in order:
        u = sweep_periodic(u, d, dt, dx, g)
    return u
