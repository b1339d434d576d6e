"""Seeded synthetic inputs and the uniform-grid harness around the hydro step.

This module serves both the tests/oracle side and the CUDA side and therefore holds NONE of the method's
arithmetic (no slopes, no predictor, no Riemann solver, no update) and imports neither the oracle nor the
CUDA binding. It knows only the problem statement: the ideal-gas variable set (R1), the array layouts of
include/gamer_hydro.h (R13), how patch groups are cut from a global box with a 2-cell ghost shell
("preparing the ghost-zone data is conducted by CPU"; R16 boundary fills) and the CFL rule
(R15: dt = C dx / max(|vx|+|vy|+|vz|+3 c_s), fp64 on the host, rounded to float32).

All randomness comes from a counter-based generator (splitmix64 -> Box-Muller) keyed by a 64-bit seed, so
every array is reproducible from (config, seed) alone. Fields are built in fp64 and rounded ONCE to
float32; that float32 array is what both the GPU and (promoted exactly) the oracle consume.

`config_3_*` is the headline workload; it STANDS IN for the paper's purely baryonic cosmological runs
(PAPER.md:29), whose initial conditions are not available: same array shapes, density contrast range,
Mach range and temperature floor as BASELINE.json:configs[3], nothing taken from any dataset.
"""
import math

import numpy as np

GAMMA = 5.0 / 3.0
N_PATCH = 16
GHOST = 2
MINMOD, VANLEER = 0, 1

# ----------------------------------------------------------------------------------------------------------
# counter-based random numbers


def _splitmix64(x):
    x = (x + np.uint64(0x9E3779B97F4A7C15)).astype(np.uint64)
    z = x
    z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
    z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
    return z ^ (z >> np.uint64(31))


def uniform01(seed, stream, n):
    """n doubles in (0,1): value i depends only on (seed, stream, i)."""
    with np.errstate(over="ignore"):
        ctr = np.arange(n, dtype=np.uint64)
        key = _splitmix64(np.array([seed], dtype=np.uint64) ^ (np.uint64(stream) * np.uint64(0xD1B54A32D192ED03)))
        z = _splitmix64(ctr ^ key)
    return ((z >> np.uint64(11)).astype(np.float64) + 0.5) * (1.0 / 9007199254740992.0)


def normal(seed, stream, n):
    """n standard normals by Box-Muller from two counter-based uniform streams."""
    m = (n + 1) // 2
    u1 = uniform01(seed, 2 * stream, m)
    u2 = uniform01(seed, 2 * stream + 1, m)
    r = np.sqrt(-2.0 * np.log(u1))
    out = np.concatenate([r * np.cos(2.0 * math.pi * u2), r * np.sin(2.0 * math.pi * u2)])
    return out[:n]


def _fft():
    try:
        import scipy.fft as sfft
        return (lambda a: sfft.rfftn(a, workers=-1)), (lambda a, s: sfft.irfftn(a, s=s, workers=-1))
    except Exception:  # pragma: no cover
        return np.fft.rfftn, (lambda a, s: np.fft.irfftn(a, s=s))


def _kgrid(n):
    k1 = np.fft.fftfreq(n, d=1.0 / n)
    kr = np.fft.rfftfreq(n, d=1.0 / n)
    return k1[:, None, None], k1[None, :, None], kr[None, None, :]


def gaussian_field(n, seed, stream, kmax, index=-2.0):
    """Periodic n^3 Gaussian random field, isotropic power P(k) ~ k^index for 1 <= |k| <= kmax, zero
    elsewhere, normalised to zero mean and unit variance. Array order [z][y][x]."""
    rfftn, irfftn = _fft()
    w = normal(seed, stream, n * n * n).reshape(n, n, n)
    wk = rfftn(w)
    kz, ky, kx = _kgrid(n)
    k2 = kx * kx + ky * ky + kz * kz
    with np.errstate(divide="ignore"):
        amp = np.where((k2 >= 1.0) & (k2 <= float(kmax) ** 2), np.power(np.maximum(k2, 1e-30), 0.25 * index), 0.0)
    f = irfftn(wk * amp, (n, n, n))
    f -= f.mean()
    f /= f.std()
    return f


# ----------------------------------------------------------------------------------------------------------
# variable set (R1)


def prim_box_to_cons(rho, vx, vy, vz, P, gamma=GAMMA):
    """[5][nz][ny][nx] conserved box (fp64) from primitive fields; E = P/(gamma-1) + 1/2 rho |v|^2."""
    U = np.empty((5,) + rho.shape, dtype=np.float64)
    U[0] = rho
    U[1] = rho * vx
    U[2] = rho * vy
    U[3] = rho * vz
    U[4] = P / (gamma - 1.0) + 0.5 * rho * (vx * vx + vy * vy + vz * vz)
    return U


def max_signal_speed(U, gamma=GAMMA):
    """max over cells of |vx|+|vy|+|vz|+3 c_s (R15), fp64. U: [...,5,nz,ny,nx]-like with variable axis -4."""
    U = np.asarray(U, dtype=np.float64)
    rho, mx, my, mz, E = (np.take(U, q, axis=-4) for q in range(5))
    P = (gamma - 1.0) * (E - 0.5 * (mx * mx + my * my + mz * mz) / rho)
    cs = np.sqrt(gamma * np.maximum(P, 0.0) / rho)
    return float(np.max((np.abs(mx) + np.abs(my) + np.abs(mz)) / rho + 3.0 * cs))


def cfl_dt(U, dx, cfl, gamma=GAMMA):
    """R15 time step, computed in fp64 and rounded to float32 (R11). Returns a Python float holding that
    float32 value."""
    return float(np.float32(cfl * dx / max_signal_speed(U, gamma)))


# ----------------------------------------------------------------------------------------------------------
# patch groups <-> global box (R13 layouts, R16 boundary fills)


def pad_box(U, bc, ghost=GHOST):
    """Ghost-fill a [5][nz][ny][nx] box. bc = (bx, by, bz), each 'periodic' or 'outflow' (copy nearest cell)."""
    mode = {"periodic": "wrap", "outflow": "edge"}
    out = U
    for axis, b in zip((3, 2, 1), bc):
        pw = [(0, 0)] * 4
        pw[axis] = (ghost, ghost)
        out = np.pad(out, pw, mode=mode[b])
    return out


def cut_groups(U, bc, N=N_PATCH, ghost=GHOST, dtype=None):
    """[5][nz][ny][nx] box -> [G][5][S][S][S] patch groups with ghost shells, group index x-fastest
    (g = (gz*Gy + gy)*Gx + gx)."""
    P = pad_box(U, bc, ghost)
    S = N + 2 * ghost
    win = np.lib.stride_tricks.sliding_window_view(P, (S, S, S), axis=(1, 2, 3))[:, ::N, ::N, ::N]
    gz, gy, gx = win.shape[1:4]
    out = np.ascontiguousarray(win.transpose(1, 2, 3, 0, 4, 5, 6), dtype=dtype or U.dtype)
    return out.reshape(gz * gy * gx, 5, S, S, S)


def assemble_box(groups_out, shape, N=N_PATCH):
    """[G][5][N][N][N] -> [5][nz][ny][nx]; inverse of cut_groups on the interiors."""
    nz, ny, nx = shape
    gz, gy, gx = nz // N, ny // N, nx // N
    a = np.asarray(groups_out).reshape(gz, gy, gx, 5, N, N, N).transpose(3, 0, 4, 1, 5, 2, 6)
    return np.ascontiguousarray(a).reshape(5, nz, ny, nx)


class Workload:
    """A global box plus everything needed to step it: U [5][nz][ny][nx] float32 (the once-rounded field),
    dx, boundary fills, limiter, CFL number, number of steps, gamma."""

    def __init__(self, name, U32, dx, bc, limiter, cfl, steps, gamma=GAMMA, meta=None):
        self.name, self.U, self.dx, self.bc = name, U32, float(dx), tuple(bc)
        self.limiter, self.cfl, self.steps, self.gamma = int(limiter), float(cfl), int(steps), float(gamma)
        self.meta = dict(meta or {})

    @property
    def shape(self):
        return self.U.shape[1:]

    @property
    def n_groups(self):
        nz, ny, nx = self.shape
        return (nz // N_PATCH) * (ny // N_PATCH) * (nx // N_PATCH)

    def groups(self, dtype=np.float32):
        return cut_groups(self.U, self.bc, dtype=dtype)

    def dt(self):
        return cfl_dt(self.U, self.dx, self.cfl, self.gamma)


def advance(U, dx, bc, limiter, cfl, steps, step_fn, gamma=GAMMA, dtype=np.float32, on_step=None):
    """Multi-step uniform-grid driver (harness, outside the hot path). Each step: dt by R15 from the current
    box -> ghost fill + cut (R16) -> step_fn(groups, dt) -> reassemble. step_fn returns U_out
    [G][5][N][N][N] (any float dtype); the box is kept in `dtype`. Returns (U, elapsed time, list of dt)."""
    U = np.asarray(U, dtype=dtype)
    t, dts = 0.0, []
    for n in range(steps):
        dt = cfl_dt(U, dx, cfl, gamma)
        out = step_fn(cut_groups(U, bc, dtype=dtype), dt)
        U = assemble_box(np.asarray(out, dtype=dtype), U.shape[1:])
        t += dt
        dts.append(dt)
        if on_step is not None:
            on_step(n, U, t)
    return U, t, dts


# ----------------------------------------------------------------------------------------------------------
# the five configurations of BASELINE.json (sizes are parameters so tests can run scaled-down versions)


def _sod_box(nx, ny, nz, axis=0, reverse=False):
    x = (np.arange((nx, ny, nz)[axis]) + 0.5) / (nx, ny, nz)[axis]
    left = x < 0.5
    if reverse:
        left = ~left
    shp = [1, 1, 1]
    shp[2 - axis] = -1
    left = np.broadcast_to(left.reshape(shp), (nz, ny, nx))
    rho = np.where(left, 1.0, 0.125)
    P = np.where(left, 1.0, 0.1)
    z = np.zeros((nz, ny, nx))
    return prim_box_to_cons(rho, z, z, z, P)


def config_0_sod3d():
    """configs[0]: 32^3 box, 2x2x2 groups, Sod step along x, outflow ghosts, MinMod, 1 step, C=0.5."""
    U = _sod_box(32, 32, 32).astype(np.float32)
    return Workload("cfg0_sod3d_8groups", U, 1.0 / 32, ("outflow",) * 3, MINMOD, 0.5, 1)


def config_1_sod_tube(nx=1024, limiter=MINMOD, steps=200, axis=0, reverse=False, dtype=np.float32):
    """configs[1]: Sod tube, 64x1x1 groups (1024x16x16), outflow along the tube, periodic across."""
    dims = [16, 16, 16]
    dims[axis] = nx
    U = _sod_box(*dims, axis=axis, reverse=reverse).astype(dtype)
    bc = ["periodic"] * 3
    bc[axis] = "outflow"
    return Workload("cfg1_sod_tube_%d" % nx, U, 1.0 / nx, bc, limiter, 0.5, steps)


def config_2_turbulence(n=256, seed=2, steps=10):
    """configs[2]: periodic n^3 (256^3 = 4096 groups), smooth turbulence, van Leer, 10 steps, C=0.5.
    ln rho ~ N(-s^2/2, s=0.5), ln P ~ N(0, 0.3), velocity components independent fields with
    rms|v| / mean(c_s) = 1; all fields P(k) ~ k^-2 for 1 <= |k| <= n/8 (>= 8 cells per shortest wave)."""
    kmax = max(2, n // 8)
    rho = np.exp(0.5 * gaussian_field(n, seed, 0, kmax) - 0.125)
    P = np.exp(0.3 * gaussian_field(n, seed, 1, kmax))
    v = [gaussian_field(n, seed, 2 + d, kmax) for d in range(3)]
    cs = np.sqrt(GAMMA * P / rho)
    scale = cs.mean() / math.sqrt(np.mean(v[0] ** 2 + v[1] ** 2 + v[2] ** 2))
    U = prim_box_to_cons(rho, v[0] * scale, v[1] * scale, v[2] * scale, P).astype(np.float32)
    return Workload("cfg2_turbulence_%d" % n, U, 1.0 / n, ("periodic",) * 3, VANLEER, 0.5, steps,
                    meta=dict(seed=seed, kmax=kmax))


def config_3_cosmo(n=512, seed=3, mach_max=30.0):
    """configs[3] (headline): periodic n^3 (512^3 = 32768 groups), cosmology-like baryonic field, MinMod,
    one step, C=0.5. rho = clip(exp(g - s^2/2), 1e-2, 1e4) with g Gaussian (s = 1.8, k^-2, |k| <= n/8);
    phi from laplacian(phi) = rho - mean; v = -s_v grad(phi), s_v set so max(|v|/c_s) = mach_max (infall
    toward the density peaks); P = rho T, T = 1e-6 max(1, rho^(gamma-1))."""
    rfftn, irfftn = _fft()
    kmax = max(2, n // 8)
    sig = 1.8
    rho = np.clip(np.exp(sig * gaussian_field(n, seed, 0, kmax) - 0.5 * sig * sig), 1e-2, 1e4)
    kz, ky, kx = _kgrid(n)
    k2 = kx * kx + ky * ky + kz * kz
    k2[0, 0, 0] = 1.0
    phik = -rfftn(rho - rho.mean()) / (k2 * (2.0 * math.pi) ** 2)
    phik[0, 0, 0] = 0.0
    tw = 2.0j * math.pi
    v = [-irfftn(tw * kk * phik, (n, n, n)) for kk in (kx, ky, kz)]
    T = 1e-6 * np.maximum(1.0, rho ** (GAMMA - 1.0))
    P = rho * T
    mach = np.sqrt(v[0] ** 2 + v[1] ** 2 + v[2] ** 2) / np.sqrt(GAMMA * T)
    s = mach_max / mach.max()
    U = prim_box_to_cons(rho, s * v[0], s * v[1], s * v[2], P).astype(np.float32)
    return Workload("cfg3_cosmo_%d" % n, U, 1.0 / n, ("periodic",) * 3, MINMOD, 0.5, 1,
                    meta=dict(seed=seed, kmax=kmax, mach_max=mach_max))


def config_4_sedov(n=256, steps=100, dtype=np.float64):
    """configs[4]: periodic n^3, rho = 1, P = 1e-5, v = 0; P = 1e5 in the cells whose centre lies within
    2 dx of the box centre (a cell corner => exactly 32 cells). MinMod, C = 0.4. meta['E0'] is the blast
    energy (sum of E dx^3 over the hot cells minus the ambient)."""
    dx = 1.0 / n
    c = (np.arange(n) + 0.5) * dx - 0.5
    r2 = c[:, None, None] ** 2 + c[None, :, None] ** 2 + c[None, None, :] ** 2
    hot = r2 <= (2.0 * dx) ** 2 * (1.0 + 1e-12)
    P = np.where(hot, 1e5, 1e-5)
    one, z = np.ones((n, n, n)), np.zeros((n, n, n))
    U = prim_box_to_cons(one, z, z, z, P).astype(dtype)
    E0 = float(hot.sum()) * (1e5 - 1e-5) / (GAMMA - 1.0) * dx ** 3
    return Workload("cfg4_sedov_%d" % n, U, dx, ("periodic",) * 3, MINMOD, 0.4, steps,
                    meta=dict(E0=E0, hot_cells=int(hot.sum())))


def random_groups(n_groups, seed, N=N_PATCH, ghost=GHOST, contrast=0.5, mach=0.7, dtype=np.float32):
    """Independent random positive states in every stored cell (not cut from a box): a stress input for
    cell-by-cell parity where every slope/limiter branch and every ghost cell is exercised."""
    S = N + 2 * ghost
    n = n_groups * S ** 3
    rho = np.exp(contrast * normal(seed, 0, n))
    P = np.exp(contrast * normal(seed, 1, n))
    cs = np.sqrt(GAMMA * P / rho)
    v = [mach * cs * normal(seed, 2 + d, n) / math.sqrt(3.0) for d in range(3)]
    U = prim_box_to_cons(rho, v[0], v[1], v[2], P)  # [5][n]
    return np.ascontiguousarray(U.reshape(5, n_groups, S, S, S).transpose(1, 0, 2, 3, 4), dtype=dtype)
