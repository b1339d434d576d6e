"""Thin Python face of the C ABI in include/gamer_hydro.h — argument marshalling only. Every step of the hot
path (reconstruction, half-step prediction, Roe solver, full-step update) runs inside
libgamer_hydro.so's CUDA kernels; PyTorch supplies device memory and streams, nothing else. There is no CPU
fallback: if the library is missing or no sm_100 device is present the calls raise.

Function names and argument order follow the C header one to one.
"""
import ctypes as C
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libgamer_hydro.so")
_lib = None

MINMOD, VANLEER, MC = 0, 1, 2
FLAG_ENTROPY_FIX, FLAG_HLLE_FALLBACK = 1, 2
PATH_AUTO, PATH_GENERIC, PATH_FUSED, PATH_FUSED_SCALAR, PATH_FUSED_DUO = 0, 1, 2, 3, 4

EXPORTS = ["gamer_hydro_alloc", "gamer_hydro_free", "gamer_hydro_step", "gamer_hydro_step_f64",
           "gamer_hydro_step_host", "gamer_hydro_status", "gamer_hydro_set_path", "gamer_hydro_launch_count",
           "gamer_hydro_strerror", "gamer_hydro_max_speed", "gamer_hydro_fill_ghosts", "gamer_hydro_advance",
           "gamer_hydro_step_grid", "gamer_hydro_set_guard_map", "gamer_rtvd_step", "gamer_hydro_step_ex", "gamer_hydro_step_ex_f64",
           "gamer_hydro_max_speed_noalloc", "gamer_hydro_max_speed_noalloc_limit", "gamer_hydro_set_hlle_map"]
BC_PERIODIC, BC_OUTFLOW = 0, 1


class GamerHydroError(RuntimeError):
    pass


def lib():
    """Loads libgamer_hydro.so (built in-tree by paper_1007_3818_b200/build.py). Fails loudly when absent."""
    global _lib
    if _lib is None:
        if not os.path.exists(_LIB_PATH):
            raise GamerHydroError("CUDA extension %s is missing: run `python -c 'import __graft_entry__ as g; "
                                  "g.build()'` (no CPU fallback exists)" % _LIB_PATH)
        L = C.CDLL(_LIB_PATH)
        vp, i, f, d = C.c_void_p, C.c_int, C.c_float, C.c_double
        L.gamer_hydro_alloc.argtypes = [i, i, i, i, i]
        L.gamer_hydro_free.restype = None
        L.gamer_hydro_step.argtypes = [vp, vp, vp, i, i, i, f, f, f, i, vp]
        L.gamer_hydro_step_f64.argtypes = [vp, vp, vp, i, i, i, d, d, d, i, vp]
        L.gamer_hydro_step_host.argtypes = [vp, vp, vp, i, i, i, f, f, f, i, i]
        L.gamer_hydro_status.argtypes = [C.POINTER(C.c_ulonglong), C.POINTER(C.c_ulonglong)]
        L.gamer_hydro_set_path.argtypes = [i]
        L.gamer_hydro_max_speed.argtypes = [vp, i, i, i, i, d, C.POINTER(C.c_double), vp]
        L.gamer_hydro_max_speed_noalloc.argtypes = [vp, i, i, i, f, vp, vp]
        L.gamer_hydro_max_speed_noalloc_limit.argtypes = []
        L.gamer_hydro_fill_ghosts.argtypes = [vp, vp, i, i, i, i, i, i, i, i, i, vp]
        L.gamer_hydro_step_grid.argtypes = [vp, vp, vp, vp, i, i, i, i, i, f, f, f, i, vp]
        L.gamer_hydro_advance.argtypes = [vp, vp, vp, i, i, i, i, i, i, i, i, i, f, f, f, i, vp, vp]
        L.gamer_hydro_set_guard_map.argtypes = [vp]
        L.gamer_hydro_set_hlle_map.argtypes = [vp]
        L.gamer_rtvd_step.argtypes = [vp, vp, i, i, i, f, f, f, i, vp]
        L.gamer_hydro_step_ex.argtypes = [vp, vp, vp, vp, i, i, i, f, f, f, i, i, vp]
        L.gamer_hydro_step_ex_f64.argtypes = [vp, vp, vp, vp, i, i, i, d, d, d, i, i, vp]
        L.gamer_hydro_launch_count.restype = C.c_ulonglong
        L.gamer_hydro_strerror.restype = C.c_char_p
        L.gamer_hydro_strerror.argtypes = [i]
        _lib = L
    return _lib


def gamer_hydro_strerror(code):
    return lib().gamer_hydro_strerror(int(code)).decode()


def _check(rc):
    if rc != 0:
        raise GamerHydroError("gamer_hydro error %d: %s" % (rc, gamer_hydro_strerror(rc)))


def gamer_hydro_alloc(max_groups, N=16, ghost=2, bytes_per_real=4, device=0):
    _check(lib().gamer_hydro_alloc(int(max_groups), int(N), int(ghost), int(bytes_per_real), int(device)))


def gamer_hydro_free():
    lib().gamer_hydro_free()


def _stream_ptr(stream):
    s = stream if stream is not None else torch.cuda.current_stream()
    return C.c_void_p(s.cuda_stream)


def _shapes(U_in, N, ghost):
    S = N + 2 * ghost
    if U_in.dim() != 5 or tuple(U_in.shape[1:]) != (5, S, S, S):
        raise GamerHydroError("U_in must be [n_groups][5][%d][%d][%d], got %s" % (S, S, S, tuple(U_in.shape)))
    return U_in.shape[0]


def _step(fn, dtype, U_in, U_out, boundary_fluxes, N, ghost, dt, dx, gamma, limiter, stream):
    G = _shapes(U_in, N, ghost)
    for x in (U_in, U_out, boundary_fluxes):
        if x is not None and not (x.is_cuda and x.dtype == dtype and x.is_contiguous()):
            raise GamerHydroError("tensors must be contiguous CUDA tensors of dtype %s" % dtype)
    if U_out is None:
        U_out = torch.empty((G, 5, N, N, N), dtype=dtype, device=U_in.device)
    if tuple(U_out.shape) != (G, 5, N, N, N):
        raise GamerHydroError("U_out must be [%d][5][%d][%d][%d], got %s" % (G, N, N, N, tuple(U_out.shape)))
    if boundary_fluxes is not None and tuple(boundary_fluxes.shape) != (G, 6, 5, N, N):
        raise GamerHydroError("boundary_fluxes must be [%d][6][5][%d][%d], got %s" % (G, N, N, tuple(boundary_fluxes.shape)))
    if any(x is not None and x.device != U_in.device for x in (U_out, boundary_fluxes)):
        raise GamerHydroError("all tensors must live on the same CUDA device")
    bf = boundary_fluxes.data_ptr() if boundary_fluxes is not None else None
    _check(fn(U_in.data_ptr(), U_out.data_ptr(), bf, G, N, ghost, dt, dx, gamma, int(limiter), _stream_ptr(stream)))
    return U_out


def gamer_hydro_step(U_in_with_ghosts, U_out, boundary_fluxes, n_groups=None, N=16, ghost=2, dt=None, dx=None,
                     gamma=5.0 / 3.0, limiter=MINMOD, stream=None):
    """fp32 step on device tensors; enqueues on `stream` (default: torch's current stream) and returns U_out."""
    assert n_groups is None or n_groups == U_in_with_ghosts.shape[0]
    return _step(lib().gamer_hydro_step, torch.float32, U_in_with_ghosts, U_out, boundary_fluxes, N, ghost, dt, dx,
                 gamma, limiter, stream)


def gamer_hydro_step_f64(U_in_with_ghosts, U_out, boundary_fluxes, n_groups=None, N=16, ghost=2, dt=None, dx=None,
                         gamma=5.0 / 3.0, limiter=MINMOD, stream=None):
    assert n_groups is None or n_groups == U_in_with_ghosts.shape[0]
    return _step(lib().gamer_hydro_step_f64, torch.float64, U_in_with_ghosts, U_out, boundary_fluxes, N, ghost, dt,
                 dx, gamma, limiter, stream)


def gamer_hydro_step_host(h_U_in, h_U_out, h_boundary_fluxes, n_groups=None, N=16, ghost=2, dt=None, dx=None,
                          gamma=5.0 / 3.0, limiter=MINMOD, chunk_groups=0):
    """fp32 step on HOST tensors (pinned recommended); copies are inside the call; synchronous."""
    G = _shapes(h_U_in, N, ghost)
    for x in (h_U_in, h_U_out, h_boundary_fluxes):
        if x is not None and (x.is_cuda or x.dtype != torch.float32 or not x.is_contiguous()):
            raise GamerHydroError("host tensors must be contiguous CPU float32 tensors")
    bf = h_boundary_fluxes.data_ptr() if h_boundary_fluxes is not None else None
    _check(lib().gamer_hydro_step_host(h_U_in.data_ptr(), h_U_out.data_ptr(), bf, G, N, ghost, dt, dx, gamma,
                                       int(limiter), int(chunk_groups)))
    return h_U_out


def _real_bytes(x):
    if not (x.is_cuda and x.is_contiguous() and x.dtype in (torch.float32, torch.float64)):
        raise GamerHydroError("tensors must be contiguous CUDA tensors of dtype float32 or float64")
    return 4 if x.dtype == torch.float32 else 8


def gamer_hydro_max_speed(U, N=16, ghost=2, gamma=5.0 / 3.0, stream=None):
    """max over the interior cells of |vx|+|vy|+|vz|+3 c_s (R15) of a device array [G][5][S][S][S]; synchronises."""
    S = N + 2 * ghost
    if U.dim() != 5 or tuple(U.shape[1:]) != (5, S, S, S):
        raise GamerHydroError("U must be [n_groups][5][%d][%d][%d]" % (S, S, S))
    out = C.c_double(0.0)
    _check(lib().gamer_hydro_max_speed(U.data_ptr(), _real_bytes(U), U.shape[0], N, ghost, gamma, C.byref(out),
                                       _stream_ptr(stream)))
    return float(out.value)


def gamer_hydro_max_speed_noalloc_limit():
    """Largest number of patch groups gamer_hydro_max_speed_noalloc takes in one call."""
    return int(lib().gamer_hydro_max_speed_noalloc_limit())


def gamer_hydro_max_speed_noalloc(U, d_max, N=16, ghost=2, gamma=5.0 / 3.0, stream=None):
    """Signal-speed maximum (R15) of a float32 device array [G][5][S][S][S] into d_max, a float32 CUDA tensor with one
    element that the caller owns. For callers that must not trigger a device allocation (an AMR code that has filled the
    GPU with its own pools; a multi-stream time loop that a device-wide cudaMalloc would stall): the library keeps the
    partial maxima in a fixed array of its own, at most gamer_hydro_max_speed_noalloc_limit() groups per call. Nothing
    is allocated here either: pass d_max in, read it back on the same stream. Enqueues and returns d_max; calls that
    could overlap on the GPU must be ordered by the caller (they share that array). Make the first call on a device
    outside any stream capture."""
    S = N + 2 * ghost
    if U.dim() != 5 or tuple(U.shape[1:]) != (5, S, S, S):
        raise GamerHydroError("U must be [n_groups][5][%d][%d][%d]" % (S, S, S))
    if not (U.is_cuda and U.dtype == torch.float32 and U.is_contiguous()):
        raise GamerHydroError("U must be a contiguous CUDA float32 tensor")
    if not (d_max.is_cuda and d_max.dtype == torch.float32 and d_max.numel() == 1 and d_max.device == U.device):
        raise GamerHydroError("d_max must be a one-element CUDA float32 tensor on the device of U")
    _check(lib().gamer_hydro_max_speed_noalloc(U.data_ptr(), U.shape[0], N, ghost, gamma, d_max.data_ptr(),
                                               _stream_ptr(stream)))
    return d_max


def gamer_hydro_fill_ghosts(U_out, U_in_with_ghosts, grid, N=16, ghost=2, bc=(BC_PERIODIC,) * 3, stream=None):
    """Rebuilds U_in_with_ghosts [G][5][S][S][S] from the interiors U_out [G][5][N][N][N] of one uniform grid of
    grid = (gx, gy, gz) groups (x-fastest group index); bc per axis: BC_PERIODIC or BC_OUTFLOW (R16)."""
    gx, gy, gz = (int(v) for v in grid)
    G, S = gx * gy * gz, N + 2 * ghost
    if tuple(U_out.shape) != (G, 5, N, N, N) or tuple(U_in_with_ghosts.shape) != (G, 5, S, S, S):
        raise GamerHydroError("shapes do not match a %dx%dx%d grid of groups" % (gx, gy, gz))
    if _real_bytes(U_out) != _real_bytes(U_in_with_ghosts):
        raise GamerHydroError("U_out and U_in_with_ghosts must have the same dtype")
    _check(lib().gamer_hydro_fill_ghosts(U_out.data_ptr(), U_in_with_ghosts.data_ptr(), _real_bytes(U_out), gx, gy, gz,
                                         N, ghost, int(bc[0]), int(bc[1]), int(bc[2]), _stream_ptr(stream)))
    return U_in_with_ghosts


def gamer_hydro_step_grid(U_with_ghosts, U_out, boundary_fluxes, U_next_with_ghosts, grid, dt, dx, N=16, ghost=2,
                          gamma=5.0 / 3.0, limiter=MINMOD, stream=None):
    """One fp32 step of a fully periodic uniform grid; the kernel also writes the next step's ghosted array."""
    gx, gy, gz = (int(v) for v in grid)
    G, S = gx * gy * gz, N + 2 * ghost
    if tuple(U_with_ghosts.shape) != (G, 5, S, S, S) or tuple(U_next_with_ghosts.shape) != (G, 5, S, S, S) or \
            tuple(U_out.shape) != (G, 5, N, N, N):
        raise GamerHydroError("shapes do not match a %dx%dx%d grid of groups" % (gx, gy, gz))
    for x in (U_with_ghosts, U_out, boundary_fluxes, U_next_with_ghosts):
        if x is not None and not (x.is_cuda and x.dtype == torch.float32 and x.is_contiguous()):
            raise GamerHydroError("tensors must be contiguous CUDA float32 tensors")
    bf = boundary_fluxes.data_ptr() if boundary_fluxes is not None else None
    _check(lib().gamer_hydro_step_grid(U_with_ghosts.data_ptr(), U_out.data_ptr(), bf, U_next_with_ghosts.data_ptr(),
                                       gx, gy, gz, N, ghost, dt, dx, gamma, int(limiter), _stream_ptr(stream)))
    return U_next_with_ghosts


def gamer_hydro_advance(U_with_ghosts, U_out, boundary_fluxes, grid, n_steps, cfl, dx, N=16, ghost=2,
                        bc=(BC_PERIODIC,) * 3, gamma=5.0 / 3.0, limiter=MINMOD, stream=None):
    """n_steps fp32 steps on one uniform grid without leaving the device; returns the list of time steps taken."""
    gx, gy, gz = (int(v) for v in grid)
    G, S = gx * gy * gz, N + 2 * ghost
    if tuple(U_with_ghosts.shape) != (G, 5, S, S, S) or tuple(U_out.shape) != (G, 5, N, N, N):
        raise GamerHydroError("shapes do not match a %dx%dx%d grid of groups" % (gx, gy, gz))
    for x in (U_with_ghosts, U_out, boundary_fluxes):
        if x is not None and not (x.is_cuda and x.dtype == torch.float32 and x.is_contiguous()):
            raise GamerHydroError("tensors must be contiguous CUDA float32 tensors")
    dts = (C.c_float * max(int(n_steps), 1))()
    bf = boundary_fluxes.data_ptr() if boundary_fluxes is not None else None
    _check(lib().gamer_hydro_advance(U_with_ghosts.data_ptr(), U_out.data_ptr(), bf, gx, gy, gz, N, ghost, int(bc[0]),
                                     int(bc[1]), int(bc[2]), int(n_steps), cfl, dx, gamma, int(limiter), dts,
                                     _stream_ptr(stream)))
    return [float(dts[s]) for s in range(int(n_steps))]


def gamer_hydro_status():
    a, b = C.c_ulonglong(0), C.c_ulonglong(0)
    _check(lib().gamer_hydro_status(C.byref(a), C.byref(b)))
    return int(a.value), int(b.value)


def gamer_hydro_set_path(path):
    _check(lib().gamer_hydro_set_path(int(path)))


def _step_ex(fn, dtype, U_in, U_out, boundary_fluxes, midplane_fluxes, N, ghost, dt, dx, gamma, limiter, flags, stream):
    G = _shapes(U_in, N, ghost)
    if U_out is None:
        U_out = torch.empty((G, 5, N, N, N), dtype=dtype, device=U_in.device)
    want = {"U_out": (U_out, (G, 5, N, N, N)), "boundary_fluxes": (boundary_fluxes, (G, 6, 5, N, N)),
            "midplane_fluxes": (midplane_fluxes, (G, 3, 5, N, N))}
    for name, (x, shape) in want.items():
        if x is None:
            continue
        if not (x.is_cuda and x.dtype == dtype and x.is_contiguous() and x.device == U_in.device):
            raise GamerHydroError("%s must be a contiguous CUDA tensor of dtype %s on the device of U_in" % (name, dtype))
        if tuple(x.shape) != shape:
            raise GamerHydroError("%s must have shape %s, got %s" % (name, shape, tuple(x.shape)))
    if not (U_in.is_cuda and U_in.dtype == dtype and U_in.is_contiguous()):
        raise GamerHydroError("U_in must be a contiguous CUDA tensor of dtype %s" % dtype)
    ptr = lambda x: x.data_ptr() if x is not None else None
    _check(fn(U_in.data_ptr(), U_out.data_ptr(), ptr(boundary_fluxes), ptr(midplane_fluxes), G, N, ghost, dt, dx, gamma,
              int(limiter), int(flags), _stream_ptr(stream)))
    return U_out


def gamer_hydro_step_ex(U_in_with_ghosts, U_out, boundary_fluxes, midplane_fluxes, n_groups=None, N=16, ghost=2, dt=None,
                        dx=None, gamma=5.0 / 3.0, limiter=MINMOD, flags=0, stream=None):
    """fp32 step with the robustness variants (MC limiter via `limiter`, FLAG_* bits, mid-plane fluxes [G][3][5][N][N])."""
    assert n_groups is None or n_groups == U_in_with_ghosts.shape[0]
    return _step_ex(lib().gamer_hydro_step_ex, torch.float32, U_in_with_ghosts, U_out, boundary_fluxes, midplane_fluxes,
                    N, ghost, dt, dx, gamma, limiter, flags, stream)


def gamer_hydro_step_ex_f64(U_in_with_ghosts, U_out, boundary_fluxes, midplane_fluxes, n_groups=None, N=16, ghost=2,
                            dt=None, dx=None, gamma=5.0 / 3.0, limiter=MINMOD, flags=0, stream=None):
    assert n_groups is None or n_groups == U_in_with_ghosts.shape[0]
    return _step_ex(lib().gamer_hydro_step_ex_f64, torch.float64, U_in_with_ghosts, U_out, boundary_fluxes,
                    midplane_fluxes, N, ghost, dt, dx, gamma, limiter, flags, stream)


def gamer_rtvd_step(U_in_with_ghosts, U_out, n_groups=None, N=16, ghost=3, dt=None, dx=None, gamma=5.0 / 3.0, sweep=0,
                    stream=None):
    """One relaxing-TVD step (fp32) on device tensors [G][5][N+2*ghost]^3 -> [G][5][N]^3; returns U_out."""
    G = _shapes(U_in_with_ghosts, N, ghost)
    assert n_groups is None or n_groups == G
    if U_out is None:
        U_out = torch.empty((G, 5, N, N, N), dtype=torch.float32, device=U_in_with_ghosts.device)
    for x in (U_in_with_ghosts, U_out):
        if not (x.is_cuda and x.dtype == torch.float32 and x.is_contiguous()):
            raise GamerHydroError("tensors must be contiguous CUDA float32 tensors")
    if tuple(U_out.shape) != (G, 5, N, N, N) or U_out.device != U_in_with_ghosts.device:
        raise GamerHydroError("U_out must be [%d][5][%d][%d][%d] on the device of U_in" % (G, N, N, N))
    _check(lib().gamer_rtvd_step(U_in_with_ghosts.data_ptr(), U_out.data_ptr(), G, N, ghost, dt, dx, gamma, int(sweep),
                                 _stream_ptr(stream)))
    return U_out


def gamer_hydro_set_guard_map(device_map):
    """device_map: zeroed uint8 CUDA tensor [n_groups][N+2][N+2][N+2], or None to switch the export off."""
    if device_map is not None and not (device_map.is_cuda and device_map.dtype == torch.uint8 and
                                       device_map.is_contiguous()):
        raise GamerHydroError("guard map must be a contiguous CUDA uint8 tensor")
    _check(lib().gamer_hydro_set_guard_map(device_map.data_ptr() if device_map is not None else None))


def gamer_hydro_set_hlle_map(device_map):
    """device_map: zeroed uint8 CUDA tensor [n_groups][3][N+1][N+1][N+1] that later gamer_hydro_step_ex calls mark with
    the faces that took the HLLE branch, or None to switch the export off."""
    if device_map is not None and not (device_map.is_cuda and device_map.dtype == torch.uint8 and
                                       device_map.is_contiguous()):
        raise GamerHydroError("HLLE map must be a contiguous CUDA uint8 tensor")
    _check(lib().gamer_hydro_set_hlle_map(device_map.data_ptr() if device_map is not None else None))


def gamer_hydro_launch_count():
    return int(lib().gamer_hydro_launch_count())
