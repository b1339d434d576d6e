"""oracle/mhm_oracle.py — ctypes face of the fp64 CPU oracle. TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs (and tests/parity_util.py) may import this.
It imports nothing from paper_1007_3818_b200 (the CUDA path) and never will. The arithmetic lives in
oracle/mhm_oracle.hpp, which cites the passages it follows (SURVEY.md §8(c) O0–O8).

Inputs given as float32 are promoted to float64 exactly (O0: "the same fp32 bits given to the GPU");
dt, dx, gamma are taken as given — callers round them to float32 first when comparing with the fp32 GPU
path (R11).
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

_lib = None

_dp = C.POINTER(C.c_double)
_u8p = C.POINTER(C.c_ubyte)
_u64p = C.POINTER(C.c_ulonglong)


def _ptr(a, typ):
    return a.ctypes.data_as(typ) if a is not None else typ()


def lib():
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(path)
        L.mhm_oracle_max_threads.restype = C.c_int
        L.mhm_oracle_step_groups.restype = C.c_int
        L.mhm_oracle_step_groups.argtypes = [_dp, C.c_int, C.c_int, C.c_int, C.c_double, C.c_double, C.c_double,
                                             C.c_int, _dp, _dp, _u8p, _dp, _u64p, C.c_int]
        L.mhm_oracle_step_box.restype = None
        L.mhm_oracle_step_box.argtypes = [_dp, C.c_int, C.c_int, C.c_int, C.c_int, C.c_double, C.c_double,
                                          C.c_double, C.c_int, _dp, _dp, _u8p, _dp, _u64p]
        L.mhm_oracle_cons_to_prim.argtypes = [_dp, C.c_double, _dp]
        L.mhm_oracle_prim_to_cons.argtypes = [_dp, C.c_double, _dp]
        L.mhm_oracle_limited_slope.restype = C.c_double
        L.mhm_oracle_limited_slope.argtypes = [C.c_double, C.c_double, C.c_int]
        L.mhm_oracle_phys_flux.argtypes = [_dp, C.c_double, C.c_int, _dp]
        L.mhm_oracle_roe_flux.argtypes = [_dp, _dp, C.c_double, C.c_int, _dp]
        L.mhm_oracle_roe_decompose.argtypes = [_dp, _dp, C.c_double, C.c_int, _dp, _dp, _dp]
        L.mhm_oracle_count_flops.argtypes = [_dp, C.c_int, C.c_int, C.c_double, C.c_double, C.c_double, C.c_int,
                                             _u64p]
        L.mhm_oracle_step_groups_ex.restype = C.c_int
        L.mhm_oracle_step_groups_ex.argtypes = [_dp, C.c_int, C.c_int, C.c_int, C.c_double, C.c_double, C.c_double,
                                                C.c_int, C.c_int, _dp, _dp, _dp, _u8p, _u64p, C.c_int, _u8p]
        L.mhm_oracle_roe_flux_ex.restype = C.c_int
        L.mhm_oracle_roe_flux_ex.argtypes = [_dp, _dp, C.c_double, C.c_int, C.c_int, _dp]
        _lib = L
    return _lib


def max_threads() -> int:
    return int(lib().mhm_oracle_max_threads())


class StepResult:
    """U_out [G][5][N][N][N], bflux [G][6][5][N][N], guard/margin [G][N+2][N+2][N+2] (index = interior+1)."""

    def __init__(self, U_out, bflux, guard, margin, guard_cells, nonpositive_out, threads):
        self.U_out, self.bflux, self.guard, self.margin = U_out, bflux, guard, margin
        self.guard_cells, self.nonpositive_out, self.threads = guard_cells, nonpositive_out, threads


def step_groups(U_in, N, ghost, dt, dx, gamma, limiter, want_bflux=True, want_guard=True, n_threads=0):
    """One MUSCL-Hancock + Roe step on a batch of patch groups. U_in [G][5][S][S][S], float32 or float64."""
    U = np.ascontiguousarray(U_in, dtype=np.float64)
    S = N + 2 * ghost
    assert U.ndim == 5 and U.shape[1:] == (5, S, S, S), U.shape
    G = U.shape[0]
    out = np.empty((G, 5, N, N, N), dtype=np.float64)
    bf = np.empty((G, 6, 5, N, N), dtype=np.float64) if want_bflux else None
    gd = np.zeros((G, N + 2, N + 2, N + 2), dtype=np.uint8) if want_guard else None
    mg = np.full((G, N + 2, N + 2, N + 2), np.nan, dtype=np.float64) if want_guard else None
    stats = np.zeros(2, dtype=np.uint64)
    used = lib().mhm_oracle_step_groups(_ptr(U, _dp), G, N, ghost, float(dt), float(dx), float(gamma), int(limiter),
                                        _ptr(out, _dp), _ptr(bf, _dp), _ptr(gd, _u8p), _ptr(mg, _dp),
                                        _ptr(stats, _u64p), int(n_threads))
    return StepResult(out, bf, gd, mg, int(stats[0]), int(stats[1]), int(used))


ENTROPY_FIX, HLLE_FALLBACK = 1, 2


def step_groups_ex(U_in, N, ghost, dt, dx, gamma, limiter, flags=0, want_midflux=False, n_threads=0, want_hlle=False):
    """step_groups with the robustness variants: limiter 2 = MC, flags = ENTROPY_FIX |
    HLLE_FALLBACK, optional mid-plane fluxes [G][3][5][N][N]. Returns (StepResult, midflux or None). With want_hlle the
    result carries .hlle, uint8 [G][3][N+1][N+1][N+1]: 1 where the face on the lower side of cell (i,j,k) along axis d
    took the HLLE branch (index [g][d][k][j][i])."""
    U = np.ascontiguousarray(U_in, dtype=np.float64)
    S = N + 2 * ghost
    assert U.ndim == 5 and U.shape[1:] == (5, S, S, S), U.shape
    G = U.shape[0]
    out = np.empty((G, 5, N, N, N), dtype=np.float64)
    bf = np.empty((G, 6, 5, N, N), dtype=np.float64)
    mf = np.empty((G, 3, 5, N, N), dtype=np.float64) if want_midflux else None
    gd = np.zeros((G, N + 2, N + 2, N + 2), dtype=np.uint8)
    stats = np.zeros(2, dtype=np.uint64)
    hl = np.zeros((G, 3, N + 1, N + 1, N + 1), dtype=np.uint8) if want_hlle else None
    used = lib().mhm_oracle_step_groups_ex(_ptr(U, _dp), G, N, ghost, float(dt), float(dx), float(gamma), int(limiter),
                                           int(flags), _ptr(out, _dp), _ptr(bf, _dp), _ptr(mf, _dp), _ptr(gd, _u8p),
                                           _ptr(stats, _u64p), int(n_threads), _ptr(hl, _u8p))
    r = StepResult(out, bf, gd, None, int(stats[0]), int(stats[1]), int(used))
    r.hlle = hl
    return r, mf


def roe_flux_ex(UL, UR, gamma, d, flags):
    """Roe flux with RiemannFlags; returns (F, used_hlle)."""
    F = np.empty(5)
    h = lib().mhm_oracle_roe_flux_ex(_ptr(_vec5(UL), _dp), _ptr(_vec5(UR), _dp), float(gamma), int(d), int(flags),
                                     _ptr(F, _dp))
    return F, bool(h)


def step_box(U_in, ghost, dt, dx, gamma, limiter):
    """One step on a single box U_in [5][nz+2g][ny+2g][nx+2g] (O8, the global form). Returns StepResult with
    U_out [5][nz][ny][nx] and bflux as a flat array (six faces, SURVEY.md §8(b) order)."""
    U = np.ascontiguousarray(U_in, dtype=np.float64)
    assert U.ndim == 4 and U.shape[0] == 5
    nz, ny, nx = (s - 2 * ghost for s in U.shape[1:])
    out = np.empty((5, nz, ny, nx), dtype=np.float64)
    bf = np.empty(10 * (nz * ny + nz * nx + ny * nx), dtype=np.float64)
    gd = np.zeros((nz + 2, ny + 2, nx + 2), dtype=np.uint8)
    mg = np.full((nz + 2, ny + 2, nx + 2), np.nan, dtype=np.float64)
    stats = np.zeros(2, dtype=np.uint64)
    lib().mhm_oracle_step_box(_ptr(U, _dp), nx, ny, nz, ghost, float(dt), float(dx), float(gamma), int(limiter),
                              _ptr(out, _dp), _ptr(bf, _dp), _ptr(gd, _u8p), _ptr(mg, _dp), _ptr(stats, _u64p))
    return StepResult(out, bf, gd, mg, int(stats[0]), int(stats[1]), 1)


def _vec5(x):
    a = np.ascontiguousarray(x, dtype=np.float64)
    assert a.shape == (5,)
    return a


def cons_to_prim(U, gamma):
    W = np.empty(5)
    lib().mhm_oracle_cons_to_prim(_ptr(_vec5(U), _dp), float(gamma), _ptr(W, _dp))
    return W


def prim_to_cons(W, gamma):
    U = np.empty(5)
    lib().mhm_oracle_prim_to_cons(_ptr(_vec5(W), _dp), float(gamma), _ptr(U, _dp))
    return U


def limited_slope(dL, dR, limiter):
    return float(lib().mhm_oracle_limited_slope(float(dL), float(dR), int(limiter)))


def phys_flux(U, gamma, d):
    F = np.empty(5)
    lib().mhm_oracle_phys_flux(_ptr(_vec5(U), _dp), float(gamma), int(d), _ptr(F, _dp))
    return F


def roe_flux(UL, UR, gamma, d):
    F = np.empty(5)
    lib().mhm_oracle_roe_flux(_ptr(_vec5(UL), _dp), _ptr(_vec5(UR), _dp), float(gamma), int(d), _ptr(F, _dp))
    return F


def roe_decompose(UL, UR, gamma, d):
    al, lam, K = np.empty(5), np.empty(5), np.empty((5, 5))
    lib().mhm_oracle_roe_decompose(_ptr(_vec5(UL), _dp), _ptr(_vec5(UR), _dp), float(gamma), int(d), _ptr(al, _dp),
                                   _ptr(lam, _dp), _ptr(K, _dp))
    return al, lam, K


def count_flops(U_in_group, N, ghost, dt, dx, gamma, limiter):
    """Algorithmic FLOPs of one step on one group: dict(add, mul, div, sqrt, minmax, total, per_cell)."""
    U = np.ascontiguousarray(U_in_group, dtype=np.float64)
    S = N + 2 * ghost
    assert U.shape == (5, S, S, S)
    c = np.zeros(5, dtype=np.uint64)
    lib().mhm_oracle_count_flops(_ptr(U, _dp), N, ghost, float(dt), float(dx), float(gamma), int(limiter),
                                 _ptr(c, _u64p))
    d = dict(zip(("add", "mul", "div", "sqrt", "minmax"), (int(x) for x in c)))
    d["total"] = int(c.sum())
    d["per_cell"] = d["total"] / float(N ** 3)
    return d
