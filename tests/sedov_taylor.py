"""Sedov-Taylor similarity constant xi0 of the spherical point blast, R(t) = xi0 (E0 t^2 / rho0)^(1/5), ideal gas
(textbook similarity solution: Sedov 1959; Landau & Lifshitz, Fluid Mechanics, par. 106). Independent of oracle/ and of
the CUDA path (scipy only); derives tests/golden/sedov_xi0.txt, which pin P15 and the cfg 4 tests use for the shock
radius (SURVEY.md Appendix A states the method: "integrating the self-similar ODEs inward from the strong-shock
conditions and normalising by the energy integral").

Similarity variables: lambda = r / R(t), with Rdot = (2/5) R / t (so that R Rddot / Rdot^2 = -3/2), and
    u = Rdot U(lambda),   rho = rho0 D(lambda),   p = rho0 Rdot^2 P(lambda).
Euler's equations in spherical symmetry become three ODEs in lambda (primes = d/dlambda):
    continuity   (U - lambda) D' + D U'                   = -2 D U / lambda
    momentum     (U - lambda) U' + P' / D                 = (3/2) U
    entropy      (U - lambda) (P' / P - gamma D' / D)     = 3
with the strong-shock jump conditions at lambda = 1:  U = P = 2 / (gamma + 1),  D = (gamma + 1) / (gamma - 1).
Energy:  E0 = int (p / (gamma-1) + rho u^2 / 2) 4 pi r^2 dr = rho0 Rdot^2 R^3 I,
         I = 4 pi int_0^1 (P / (gamma-1) + D U^2 / 2) lambda^2 dlambda,
and with Rdot = (2/5) R / t and R = xi0 (E0 t^2 / rho0)^(1/5):  xi0 = (25 / (4 I))^(1/5).
"""
import math

import numpy as np
from scipy.integrate import solve_ivp


def _rhs(s, y, g):
    """Independent variable s = ln(lambda); unknowns w = U / lambda, ln D, ln P and the running energy integral.
    With a = w - 1 and T = P / (D lambda^2) the three equations of the header read (dots = d/ds)
        a (lnD). + w.              = -3 w
        a w.     + T (lnP).        = (3/2) w - a w
        a ((lnP). - gamma (lnD).)  = 3
    — every coefficient is of order one except T, which grows towards the centre where the density vanishes."""
    w, lnD, lnP, _ = y
    lam = math.exp(s)
    D, P = math.exp(lnD), math.exp(lnP)
    a, T = w - 1.0, P / (D * lam * lam)
    A = np.array([[1.0, a, 0.0],
                  [a, 0.0, T],
                  [0.0, -g * a, a]])
    b = np.array([-3.0 * w, 1.5 * w - a * w, 3.0])
    dw, dlnD, dlnP = np.linalg.solve(A, b)
    dI = 4.0 * math.pi * (P / (g - 1.0) + 0.5 * D * (w * lam) ** 2) * lam ** 3
    return [dw, dlnD, dlnP, dI]


def profiles(gamma, lam_min=1e-3, rtol=1e-10):
    """Integrates inward from the shock (s = 0) to s = ln(lam_min). Returns scipy's solution object; columns of .y are
    (U / lambda, ln D, ln P, -energy integral from lambda to 1)."""
    y0 = [2.0 / (gamma + 1.0), math.log((gamma + 1.0) / (gamma - 1.0)), math.log(2.0 / (gamma + 1.0)), 0.0]
    sol = solve_ivp(_rhs, (0.0, math.log(lam_min)), y0, args=(gamma,), method="Radau", rtol=rtol, atol=1e-12)
    assert sol.success, sol.message
    return sol


def xi0(gamma, lam_min=1e-3):
    """Similarity constant. Inside lam_min the density has fallen to ~ lam^(3/(gamma-1)) of its shock value and the
    pressure is flat, so the remaining energy is the thermal energy of a uniform-pressure ball."""
    sol = profiles(gamma, lam_min)
    _, _, lnP, J = sol.y[:, -1]
    I = -J + 4.0 * math.pi * math.exp(lnP) / (gamma - 1.0) * lam_min ** 3 / 3.0
    return (25.0 / (4.0 * I)) ** 0.2


if __name__ == "__main__":
    for name, g in (("gamma_5_3", 5.0 / 3.0), ("gamma_1_4", 1.4)):
        print("%s  %.6f" % (name, xi0(g)))
