"""Exact solution of the 1-D Riemann problem for an ideal gas (textbook closed form: pressure function +
root find + wave sampling, Toro 2009 ch. 4). Independent of oracle/ and of the CUDA path; used to pin the
oracle (P9) and to check the GPU Sod runs. tests/golden/sod_exact_gamma53.txt holds the star-state
constants quoted in SURVEY.md Appendix A, which test_oracle_pins.py checks this solver against."""
import math

import numpy as np


def _f(p, rk, pk, ck, g):
    if p > pk:  # shock
        A = 2.0 / ((g + 1.0) * rk)
        B = (g - 1.0) / (g + 1.0) * pk
        return (p - pk) * math.sqrt(A / (p + B))
    return 2.0 * ck / (g - 1.0) * ((p / pk) ** ((g - 1.0) / (2.0 * g)) - 1.0)  # rarefaction


def star_state(g, rl, ul, pl, rr, ur, pr):
    cl, cr = math.sqrt(g * pl / rl), math.sqrt(g * pr / rr)
    lo, hi = 1e-14, 10.0 * max(pl, pr)
    F = lambda p: _f(p, rl, pl, cl, g) + _f(p, rr, pr, cr, g) + ur - ul
    for _ in range(200):  # bisection: monotone function, no derivative needed
        mid = 0.5 * (lo + hi)
        if F(mid) > 0.0:
            hi = mid
        else:
            lo = mid
    ps = 0.5 * (lo + hi)
    us = 0.5 * (ul + ur) + 0.5 * (_f(ps, rr, pr, cr, g) - _f(ps, rl, pl, cl, g))
    return ps, us


def sample(g, left, right, xi):
    """Primitive solution (rho, u, p) at similarity coordinates xi = x/t (array)."""
    rl, ul, pl = left
    rr, ur, pr = right
    cl, cr = math.sqrt(g * pl / rl), math.sqrt(g * pr / rr)
    ps, us = star_state(g, rl, ul, pl, rr, ur, pr)
    xi = np.asarray(xi, dtype=np.float64)
    rho, u, p = np.empty_like(xi), np.empty_like(xi), np.empty_like(xi)
    gm = (g - 1.0) / (g + 1.0)
    for n, s in enumerate(xi.ravel()):
        if s <= us:  # left of contact
            if ps > pl:  # left shock
                q = ps / pl
                S = ul - cl * math.sqrt((g + 1.0) / (2.0 * g) * q + (g - 1.0) / (2.0 * g))
                val = (rl, ul, pl) if s <= S else (rl * (q + gm) / (gm * q + 1.0), us, ps)
            else:
                csl = cl * (ps / pl) ** ((g - 1.0) / (2.0 * g))
                if s <= ul - cl:
                    val = (rl, ul, pl)
                elif s >= us - csl:
                    val = (rl * (ps / pl) ** (1.0 / g), us, ps)
                else:
                    c = 2.0 / (g + 1.0) * (cl + 0.5 * (g - 1.0) * (ul - s))
                    val = (rl * (c / cl) ** (2.0 / (g - 1.0)), 2.0 / (g + 1.0) * (cl + 0.5 * (g - 1.0) * ul + s),
                           pl * (c / cl) ** (2.0 * g / (g - 1.0)))
        else:
            if ps > pr:  # right shock
                q = ps / pr
                S = ur + cr * math.sqrt((g + 1.0) / (2.0 * g) * q + (g - 1.0) / (2.0 * g))
                val = (rr, ur, pr) if s >= S else (rr * (q + gm) / (gm * q + 1.0), us, ps)
            else:
                csr = cr * (ps / pr) ** ((g - 1.0) / (2.0 * g))
                if s >= ur + cr:
                    val = (rr, ur, pr)
                elif s <= us + csr:
                    val = (rr * (ps / pr) ** (1.0 / g), us, ps)
                else:
                    c = 2.0 / (g + 1.0) * (cr - 0.5 * (g - 1.0) * (ur - s))
                    val = (rr * (c / cr) ** (2.0 / (g - 1.0)), 2.0 / (g + 1.0) * (-cr + 0.5 * (g - 1.0) * ur + s),
                           pr * (c / cr) ** (2.0 * g / (g - 1.0)))
        rho.flat[n], u.flat[n], p.flat[n] = val
    return rho, u, p


def sod_constants(g):
    """Star-region constants of the Sod problem (1,0,1 | 0.125,0,0.1) for comparison with the golden file."""
    rl, ul, pl, rr, ur, pr = 1.0, 0.0, 1.0, 0.125, 0.0, 0.1
    ps, us = star_state(g, rl, ul, pl, rr, ur, pr)
    cl, cr = math.sqrt(g * pl / rl), math.sqrt(g * pr / rr)
    gm = (g - 1.0) / (g + 1.0)
    q = ps / pr
    return dict(p_star=ps, u_star=us, rho_star_L=rl * (ps / pl) ** (1.0 / g),
                rho_star_R=rr * (q + gm) / (gm * q + 1.0),
                shock_speed=ur + cr * math.sqrt((g + 1.0) / (2.0 * g) * q + (g - 1.0) / (2.0 * g)),
                raref_head=ul - cl, raref_tail=us - cl * (ps / pl) ** ((g - 1.0) / (2.0 * g)))
