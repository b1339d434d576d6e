"""Error metric of reading R14: err = |g - o| / s per cell and variable, with s = |o| for
rho and E, and s = rho_o (|v_o| + c_o) for each momentum component (a component can be exactly 0). Boundary
fluxes use the flux scale rho (|v|+c) * {1, (|v|+c), (|v|+c), (|v|+c), (|v|+c)^2} of the adjacent cell."""
import numpy as np


def _scales(o, gamma):
    rho, mx, my, mz, E = (o[..., q, :, :, :] for q in range(5))
    vv = (mx * mx + my * my + mz * mz) / (rho * rho)
    P = (gamma - 1.0) * (E - 0.5 * rho * vv)
    c = np.sqrt(gamma * np.maximum(P, 0.0) / rho)
    return rho, E, np.sqrt(vv) + c


def cell_errors(g, o, gamma):
    """g, o: [...,5,N,N,N]; returns per-cell-per-variable relative error array (same shape), fp64."""
    g = np.asarray(g, dtype=np.float64)
    o = np.asarray(o, dtype=np.float64)
    rho, E, a = _scales(o, gamma)
    s = np.empty_like(o)
    s[..., 0, :, :, :] = np.abs(rho)
    s[..., 4, :, :, :] = np.abs(E)
    for q in (1, 2, 3):
        s[..., q, :, :, :] = rho * a
    return np.abs(g - o) / s


def max_rel_err(g, o, gamma, mask=None):
    e = cell_errors(g, o, gamma)
    if mask is not None:
        e = np.where(mask, e, 0.0)
    return float(np.max(e)) if e.size else 0.0


def bflux_errors(gb, ob, U_out_o, gamma):
    """gb, ob: [G,6,5,N,N]; scale from the oracle's updated interior cell adjacent to each face."""
    gb = np.asarray(gb, dtype=np.float64)
    ob = np.asarray(ob, dtype=np.float64)
    o = np.asarray(U_out_o, dtype=np.float64)
    rho, E, a = _scales(o, gamma)  # [G,N,N,N] indexed [k][j][i]
    adj = [(Ellipsis, 0), (Ellipsis, -1)]
    sl = {0: lambda x: x[:, :, :, 0], 1: lambda x: x[:, :, :, -1], 2: lambda x: x[:, :, 0, :], 3: lambda x: x[:, :, -1, :],
          4: lambda x: x[:, 0, :, :], 5: lambda x: x[:, -1, :, :]}
    err = np.empty_like(ob)
    for f in range(6):
        r, s = sl[f](rho), sl[f](a)
        base = r * s
        sc = [base, base * s, base * s, base * s, base * s * s]
        for q in range(5):
            err[:, f, q] = np.abs(gb[:, f, q] - ob[:, f, q]) / sc[q]
    del adj
    return err


NEAR_GUARD = 1e-5        # |internal/total energy| of the worst predicted face state below which fp32 may flip R7


def suspect_mask(margin, N=16):
    """Interior cells whose update can be touched by an fp32/fp64 disagreement on the R7 guard: cells whose
    own or a face neighbour's guard margin (an array the reference side provides, [G,N+2,N+2,N+2]) is within
    NEAR_GUARD of zero. Pure array logic: no method arithmetic."""
    near = np.abs(margin) < NEAR_GUARD          # NaN (cells outside R) compares False
    m = near.copy()
    m[:, 1:] |= near[:, :-1]; m[:, :-1] |= near[:, 1:]
    m[:, :, 1:] |= near[:, :, :-1]; m[:, :, :-1] |= near[:, :, 1:]
    m[:, :, :, 1:] |= near[:, :, :, :-1]; m[:, :, :, :-1] |= near[:, :, :, 1:]
    return m[:, 1:-1, 1:-1, 1:-1]
