"""oracle/rtvd_oracle.py — ctypes face of the fp64 relaxing-TVD oracle (oracle/rtvd_oracle.hpp). TEST
INFRASTRUCTURE, NOT PRODUCT CODE: only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline legs may import it;
it imports nothing from paper_1007_3818_b200. float32 inputs are promoted to float64 exactly; dt, dx, gamma are taken
as given."""
import ctypes as C

import numpy as np

from . import build as _build

_lib = None
_dp = C.POINTER(C.c_double)


def _ptr(a):
    return a.ctypes.data_as(_dp)


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build_rtvd())
        L.rtvd_oracle_step_groups.restype = C.c_int
        L.rtvd_oracle_step_groups.argtypes = [_dp, C.c_int, C.c_int, C.c_double, C.c_double, C.c_double, C.c_int, _dp,
                                              C.c_int]
        L.rtvd_oracle_step_box.restype = None
        L.rtvd_oracle_step_box.argtypes = [_dp, C.c_int, C.c_int, C.c_int, C.c_double, C.c_double, C.c_double, C.c_int,
                                           _dp]
        L.rtvd_oracle_sweep_line.restype = None
        L.rtvd_oracle_sweep_line.argtypes = [_dp, C.c_int, C.c_int, C.c_double, C.c_double, C.c_double]
        L.rtvd_oracle_vanleer.restype = C.c_double
        L.rtvd_oracle_vanleer.argtypes = [C.c_double, C.c_double]
        L.rtvd_oracle_flux_and_speed.restype = None
        L.rtvd_oracle_flux_and_speed.argtypes = [_dp, C.c_int, C.c_double, _dp, _dp]
        L.rtvd_oracle_count_flops.restype = None
        L.rtvd_oracle_count_flops.argtypes = [_dp, C.c_int, C.c_double, C.c_double, C.c_double, C.c_int,
                                              C.POINTER(C.c_ulonglong)]
        _lib = L
    return _lib


def count_flops(U_in, N, dt, dx, gamma, sweep):
    """Algorithmic FLOPs of one step on ONE group U_in [5][N+6][N+6][N+6]: the oracle text run with a counting scalar
    (oracle/counting_real.hpp). Returns dict(add, mul, div, sqrt, minmax, total, per_cell); per_cell = total / N^3."""
    U = np.ascontiguousarray(U_in, dtype=np.float64)
    assert U.shape == (5, N + 6, N + 6, N + 6), U.shape
    c = (C.c_ulonglong * 5)()
    lib().rtvd_oracle_count_flops(_ptr(U), N, float(dt), float(dx), float(gamma), int(sweep), c)
    d = dict(zip(("add", "mul", "div", "sqrt", "minmax"), (int(v) for v in c)))
    d["total"] = sum(d.values())
    d["per_cell"] = d["total"] / float(N ** 3)
    return d


def step_groups(U_in, N, dt, dx, gamma, sweep, n_threads=0):
    """One relaxing-TVD step on patch groups. U_in [G][5][N+6][N+6][N+6] -> (U_out [G][5][N][N][N], threads used)."""
    U = np.ascontiguousarray(U_in, dtype=np.float64)
    S = N + 6
    assert U.ndim == 5 and U.shape[1:] == (5, S, S, S), U.shape
    out = np.empty((U.shape[0], 5, N, N, N), dtype=np.float64)
    used = lib().rtvd_oracle_step_groups(_ptr(U), U.shape[0], N, float(dt), float(dx), float(gamma), int(sweep),
                                         _ptr(out), int(n_threads))
    return out, int(used)


def step_box(U_in, dt, dx, gamma, sweep):
    """One step on a single box U_in [5][nz+6][ny+6][nx+6] -> U_out [5][nz][ny][nx]."""
    U = np.ascontiguousarray(U_in, dtype=np.float64)
    assert U.ndim == 4 and U.shape[0] == 5
    nz, ny, nx = (s - 6 for s in U.shape[1:])
    out = np.empty((5, nz, ny, nx), dtype=np.float64)
    lib().rtvd_oracle_step_box(_ptr(U), nx, ny, nz, float(dt), float(dx), float(gamma), int(sweep), _ptr(out))
    return out


def sweep_line(u, d, dt, dx, gamma):
    """One sweep of one line u [L][5] along axis d; returns the updated copy (cells 3 .. L-4 change)."""
    v = np.ascontiguousarray(u, dtype=np.float64).copy()
    assert v.ndim == 2 and v.shape[1] == 5
    lib().rtvd_oracle_sweep_line(_ptr(v), v.shape[0], int(d), float(dt), float(dx), float(gamma))
    return v


def vanleer(a, b):
    return float(lib().rtvd_oracle_vanleer(float(a), float(b)))


def flux_and_speed(u, d, gamma):
    uu = np.ascontiguousarray(u, dtype=np.float64)
    F, c = np.empty(5), np.empty(1)
    lib().rtvd_oracle_flux_and_speed(_ptr(uu), int(d), float(gamma), _ptr(F), _ptr(c))
    return F, float(c[0])
