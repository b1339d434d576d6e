"""GPU tests (-m gpu) of the steps either side of the hot path: the CFL signal-speed
maximum (R15), the same-level ghost-shell refill (R16) and the device-resident multi-step driver. References: the
numpy harness of harness/workloads.py (pure data movement / the R15 formula in fp64) and, for the
multi-step run, the fp64 oracle stepped with the time steps the device reports."""
import numpy as np
import pytest
import torch

from harness import metrics
import parity_util as pu
import paper_1007_3818_b200 as gh
from oracle import mhm_oracle as O
from harness import workloads as wl

pytestmark = pytest.mark.gpu
G = wl.GAMMA
DEV = "cuda:0"
BC = {"periodic": gh.BC_PERIODIC, "outflow": gh.BC_OUTFLOW}


def _grid(shape):
    nz, ny, nx = shape
    return (nx // 16, ny // 16, nz // 16)


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
@pytest.mark.parametrize("bc", [("periodic",) * 3, ("outflow", "periodic", "outflow"), ("outflow",) * 3])
def test_fill_ghosts_is_the_harness_ghost_fill_bit_for_bit(bc, dtype):
    rng = np.random.default_rng(11)
    shape = (32, 48, 64)                                    # nz, ny, nx -> 2 x 3 x 4 groups
    U = rng.standard_normal((5,) + shape).astype(dtype)
    want = wl.cut_groups(U, bc)                             # [G][5][20][20][20]
    interiors = np.ascontiguousarray(want[:, :, 2:-2, 2:-2, 2:-2])
    d_out = torch.from_numpy(interiors).to(DEV)
    d_in = torch.full(want.shape, float("nan"), dtype=d_out.dtype, device=DEV)
    gh.gamer_hydro_fill_ghosts(d_out, d_in, _grid(shape), bc=[BC[b] for b in bc])
    torch.cuda.synchronize()
    assert np.array_equal(d_in.cpu().numpy(), want)
    # wider shell (ghost = 3) and a small patch size (N = 8)
    want3 = wl.cut_groups(U[:, :16, :16, :24], bc, N=8, ghost=3)
    d_out3 = torch.from_numpy(np.ascontiguousarray(want3[:, :, 3:-3, 3:-3, 3:-3])).to(DEV)
    d_in3 = torch.empty(want3.shape, dtype=d_out.dtype, device=DEV)
    gh.gamer_hydro_fill_ghosts(d_out3, d_in3, (3, 2, 2), N=8, ghost=3, bc=[BC[b] for b in bc])
    torch.cuda.synchronize()
    assert np.array_equal(d_in3.cpu().numpy(), want3)


def test_max_speed_matches_the_fp64_formula():
    w = wl.config_3_cosmo(64, seed=9)
    grp = w.groups()
    ref = wl.max_signal_speed(w.U)
    got = gh.gamer_hydro_max_speed(torch.from_numpy(grp).to(DEV))
    assert abs(got - ref) <= 1e-4 * ref, (got, ref)          # Mach-30 cells: P from a cancelling difference in fp32
    got64 = gh.gamer_hydro_max_speed(torch.from_numpy(grp.astype(np.float64)).to(DEV))
    assert abs(got64 - ref) <= 1e-12 * ref
    # interiors without ghost shells (a U_out array), fp32 on a smooth field
    w2 = wl.config_2_turbulence(64, seed=4)
    inter = np.ascontiguousarray(w2.groups()[:, :, 2:-2, 2:-2, 2:-2])
    got2 = gh.gamer_hydro_max_speed(torch.from_numpy(inter).to(DEV), ghost=0)
    ref2 = wl.max_signal_speed(w2.U)
    assert abs(got2 - ref2) <= 2e-6 * ref2
    # ghost cells must not enter the maximum
    poisoned = grp.copy()
    poisoned[:, 1:4, :2] = 1e6
    assert gh.gamer_hydro_max_speed(torch.from_numpy(poisoned).to(DEV)) == got


@pytest.mark.parametrize("path", [gh.PATH_AUTO, gh.PATH_FUSED_DUO])
@pytest.mark.parametrize("cfg", ["turbulence", "sod_tube"])
def test_device_resident_advance_matches_host_driven_steps_and_the_oracle(cfg, path):
    """gamer_hydro_advance on the default path (step + ghost refill) and on the DUO path (on a periodic grid: the
    fused-halo step kernel) against host-driven steps through the same kernel path (bit-identical) and the oracle."""
    if cfg == "turbulence":
        w, steps = wl.config_2_turbulence(64, seed=2, steps=10), 10
    else:
        w, steps = wl.config_1_sod_tube(nx=256, steps=10), 10
    grid, bc = _grid(w.shape), [BC[b] for b in w.bc]
    dx = pu.f32(w.dx)
    d_U = torch.from_numpy(w.groups()).to(DEV)
    n = d_U.shape[0]
    d_out = torch.empty((n, 5, 16, 16, 16), dtype=torch.float32, device=DEV)
    d_bf = torch.empty((n, 6, 5, 16, 16), dtype=torch.float32, device=DEV)
    gh.gamer_hydro_set_path(path)
    try:
        dts = gh.gamer_hydro_advance(d_U, d_out, d_bf, grid, steps, w.cfl, dx, bc=bc, limiter=w.limiter)
        torch.cuda.synchronize()
    finally:
        gh.gamer_hydro_set_path(gh.PATH_AUTO)
    assert len(dts) == steps and all(dt > 0 for dt in dts)
    # the harness' fp64 time step on the initial box agrees with the device's first one
    assert abs(dts[0] - wl.cfl_dt(w.U, w.dx, w.cfl)) <= 2e-6 * dts[0]
    # (1) host-driven loop through the plain step call with the same dt sequence: bit-identical
    U = w.U.copy()
    for dt in dts:
        out = pu.run_gpu(wl.cut_groups(U, w.bc), dt, dx, G, w.limiter, want_bflux=False, path=path)[0]
        U = wl.assemble_box(out, w.shape)
    assert np.array_equal(d_out.cpu().numpy(), out)
    assert np.array_equal(d_U.cpu().numpy(), wl.cut_groups(U, w.bc))       # ghost shells refilled for the next step
    # (2) the fp64 oracle with the same dt sequence: north_star's 10-step tolerance
    Uo = w.U.astype(np.float64)
    for dt in dts:
        r = O.step_groups(wl.cut_groups(Uo, w.bc), 16, 2, dt, dx, G, w.limiter, want_bflux=False, want_guard=False)
        Uo = wl.assemble_box(r.U_out, w.shape)
    assert metrics.max_rel_err(U[None], Uo[None], G) <= 1e-3


def test_advance_argument_errors():
    d_U = torch.ones((1, 5, 20, 20, 20), dtype=torch.float32, device=DEV)
    d_out = torch.empty((1, 5, 16, 16, 16), dtype=torch.float32, device=DEV)
    with pytest.raises(gh.GamerHydroError):
        gh.gamer_hydro_advance(d_U, d_out, None, (1, 1, 1), 1, -0.5, 1.0)           # cfl <= 0
    with pytest.raises(gh.GamerHydroError):
        gh.gamer_hydro_advance(d_U, d_out, None, (2, 1, 1), 1, 0.5, 1.0)            # shapes do not match the grid
    with pytest.raises(gh.GamerHydroError):
        gh.gamer_hydro_fill_ghosts(d_out, d_U, (1, 1, 1), bc=(0, 2, 0))             # unknown boundary code
    d_U[:, 1:4] = 0.0
    d_U[:, 0] = float("nan")                                                        # no finite signal speed
    with pytest.raises(gh.GamerHydroError):
        gh.gamer_hydro_advance(d_U, d_out, None, (1, 1, 1), 1, 0.5, 1.0)


@pytest.mark.parametrize("shape,limiter", [((16, 16, 16), 0), ((16, 32, 48), 1), ((64, 64, 64), 0)])
def test_fused_halo_step_equals_step_plus_ghost_refill(shape, limiter):
    """gamer_hydro_step_grid: the step kernel that writes the next step's ghosted array itself gives the same bits as
    gamer_hydro_step followed by gamer_hydro_fill_ghosts — also on grids of one or two groups per axis, where a group
    is its own periodic neighbour — and the same U_out / boundary fluxes."""
    rng = np.random.default_rng(5)
    nz, ny, nx = shape
    rho = np.exp(0.3 * rng.standard_normal(shape))
    v = 0.4 * rng.standard_normal((3,) + shape)
    P = np.exp(0.2 * rng.standard_normal(shape))
    U = wl.prim_box_to_cons(rho, v[0], v[1], v[2], P).astype(np.float32)
    bc = ("periodic",) * 3
    grid = _grid(shape)
    grp = wl.cut_groups(U, bc)
    n = grp.shape[0]
    dx = pu.f32(1.0 / nx)
    dt = wl.cfl_dt(U, 1.0 / nx, 0.4)
    d_in = torch.from_numpy(np.array(grp)).to(DEV)
    outs = []
    for fused in (False, True):
        d_out = torch.full((n, 5, 16, 16, 16), float("nan"), dtype=torch.float32, device=DEV)
        d_bf = torch.full((n, 6, 5, 16, 16), float("nan"), dtype=torch.float32, device=DEV)
        d_next = torch.full(grp.shape, float("nan"), dtype=torch.float32, device=DEV)
        if fused:
            gh.gamer_hydro_step_grid(d_in, d_out, d_bf, d_next, grid, dt, dx, limiter=limiter)
        else:
            gh.gamer_hydro_set_path(gh.PATH_FUSED_DUO)      # the fused-halo kernel is the DUO kernel with HALO = true
            try:
                gh.gamer_hydro_step(d_in, d_out, d_bf, n, 16, 2, dt, dx, G, limiter)
            finally:
                gh.gamer_hydro_set_path(gh.PATH_AUTO)
            gh.gamer_hydro_fill_ghosts(d_out, d_next, grid)
        torch.cuda.synchronize()
        outs.append((d_out.cpu().numpy(), d_bf.cpu().numpy(), d_next.cpu().numpy()))
    for a, b in zip(outs[0], outs[1]):
        assert np.isfinite(b).all()
        assert np.array_equal(a, b)
    # and the next ghosted array is what the harness builds from the interiors
    assert np.array_equal(outs[1][2], wl.cut_groups(wl.assemble_box(outs[1][0], shape), bc))
    with pytest.raises(gh.GamerHydroError):
        gh.gamer_hydro_step_grid(d_in, d_out, d_bf, d_in, grid, dt, dx)        # U_next aliases the input


@pytest.mark.parametrize("path", [gh.PATH_AUTO, gh.PATH_FUSED_DUO])
def test_advance_odd_and_even_step_counts_on_a_periodic_grid(path):
    """The fused-halo loop (DUO path) ping-pongs between the caller's array and the library's: the caller's array must
    hold the final ghosted state for odd and even step counts alike; the default path refills in place."""
    w = wl.config_2_turbulence(32, seed=7)
    grid, bc = _grid(w.shape), [BC[b] for b in w.bc]
    dx = pu.f32(w.dx)
    for steps in (1, 2, 3):
        d_U = torch.from_numpy(w.groups()).to(DEV)
        n = d_U.shape[0]
        d_out = torch.empty((n, 5, 16, 16, 16), dtype=torch.float32, device=DEV)
        gh.gamer_hydro_set_path(path)
        try:
            dts = gh.gamer_hydro_advance(d_U, d_out, None, grid, steps, w.cfl, dx, bc=bc, limiter=w.limiter)
            torch.cuda.synchronize()
        finally:
            gh.gamer_hydro_set_path(gh.PATH_AUTO)
        U = w.U.copy()
        for dt in dts:
            out = pu.run_gpu(wl.cut_groups(U, w.bc), dt, dx, G, w.limiter, want_bflux=False, path=path)[0]
            U = wl.assemble_box(out, w.shape)
        assert np.array_equal(d_out.cpu().numpy(), out)
        assert np.array_equal(d_U.cpu().numpy(), wl.cut_groups(U, w.bc)), steps


def test_fused_halo_step_on_the_guard_heavy_cosmo_field():
    """Same equality on the Mach-30 field of configs[3] (64^3), where the positivity guard fires in many cells."""
    w = wl.config_3_cosmo(64, seed=3)
    grp = np.array(w.groups())
    n, grid = grp.shape[0], _grid(w.shape)
    dt, dx = pu.f32(w.dt()), pu.f32(w.dx)
    d_in = torch.from_numpy(grp).to(DEV)
    res = []
    for fused in (False, True):
        d_out = torch.full((n, 5, 16, 16, 16), float("nan"), dtype=torch.float32, device=DEV)
        d_next = torch.full(grp.shape, float("nan"), dtype=torch.float32, device=DEV)
        gh.gamer_hydro_status()
        if fused:
            gh.gamer_hydro_step_grid(d_in, d_out, None, d_next, grid, dt, dx, limiter=w.limiter)
        else:
            gh.gamer_hydro_set_path(gh.PATH_FUSED_DUO)
            try:
                gh.gamer_hydro_step(d_in, d_out, None, n, 16, 2, dt, dx, G, w.limiter)
            finally:
                gh.gamer_hydro_set_path(gh.PATH_AUTO)
            gh.gamer_hydro_fill_ghosts(d_out, d_next, grid)
        torch.cuda.synchronize()
        res.append((d_out.cpu().numpy(), d_next.cpu().numpy(), gh.gamer_hydro_status()))
    assert res[0][2] == res[1][2] and res[0][2][0] > 0          # same guard / non-positive counts, guard active
    assert np.array_equal(res[0][0], res[1][0]) and np.array_equal(res[0][1], res[1][1])
    # the signal-speed maximum the fused kernel leaves for the next step is the maximum of the new state
    gh.gamer_hydro_set_path(gh.PATH_FUSED_DUO)
    try:
        dts = gh.gamer_hydro_advance(torch.from_numpy(grp).to(DEV), torch.empty((n, 5, 16, 16, 16), device=DEV), None,
                                     grid, 2, 0.5, dx, limiter=w.limiter)
    finally:
        gh.gamer_hydro_set_path(gh.PATH_AUTO)
    vnew = gh.gamer_hydro_max_speed(torch.from_numpy(res[1][0]).to(DEV), ghost=0)
    # (advance's first step used its own dt, so only check the relation dt = cfl dx / vmax on the second step loosely)
    assert dts[1] > 0 and np.isfinite(vnew)


def test_two_advance_loops_on_two_streams_give_the_single_stream_bits():
    """SURVEY.md 8(b) 're-entrant across streams': two gamer_hydro_advance loops (different grids, different streams,
    two host threads — ctypes releases the GIL inside the call) running concurrently give the bits of the same loops run
    one after the other: every call reduces its signal-speed maximum in its own slot."""
    import threading
    ws = [wl.config_2_turbulence(64, seed=21, steps=8), wl.config_3_cosmo(64, seed=22)]
    steps = 8

    def run(w, stream, out):
        with torch.cuda.stream(stream):
            d_U = torch.from_numpy(w.groups()).to(DEV)
            d_out = torch.empty((d_U.shape[0], 5, 16, 16, 16), dtype=torch.float32, device=DEV)
            dts = gh.gamer_hydro_advance(d_U, d_out, None, _grid(w.shape), steps, 0.4, pu.f32(w.dx),
                                         bc=[BC[b] for b in w.bc], limiter=w.limiter, stream=stream)
            stream.synchronize()
            out.append((dts, d_out.cpu().numpy(), d_U.cpu().numpy()))

    serial = [[], []]
    for k, w in enumerate(ws):
        run(w, torch.cuda.Stream(), serial[k])
    for rep in range(3):
        conc = [[], []]
        th = [threading.Thread(target=run, args=(w, torch.cuda.Stream(), conc[k])) for k, w in enumerate(ws)]
        for t in th:
            t.start()
        for t in th:
            t.join()
        for k in range(2):
            assert conc[k][0][0] == serial[k][0][0]                              # same dt sequence
            assert np.array_equal(conc[k][0][1], serial[k][0][1]) and np.array_equal(conc[k][0][2], serial[k][0][2])


def test_advance_reports_a_nan_state_and_leaves_the_completed_steps_in_U():
    w = wl.config_2_turbulence(32, seed=23)
    d_U = torch.from_numpy(w.groups()).to(DEV)
    n = d_U.shape[0]
    d_out = torch.empty((n, 5, 16, 16, 16), dtype=torch.float32, device=DEV)
    d_U[3, 4, 9, 9, 9] = float("nan")                      # one interior cell: the device maximum must become NaN
    with pytest.raises(gh.GamerHydroError):
        gh.gamer_hydro_advance(d_U, d_out, None, _grid(w.shape), 3, 0.4, pu.f32(w.dx), limiter=w.limiter)
    assert np.isnan(gh.gamer_hydro_max_speed(d_U))


def test_advance_keeps_its_reduction_slot_while_another_thread_reduces_hundreds_of_times():
    """the reduction slots used to be handed out round robin modulo 64 with no owner, so 64 calls of
    gamer_hydro_max_speed on another thread wrapped around onto the slot a running gamer_hydro_advance kept for all its
    steps (zeroed it, or added a foreign maximum: wrong dt). Slots are now leased for the duration of the call. A
    12-step advance on a cold field (maximum ~ 0.16) runs beside 400 max_speed calls on a hot field (maximum ~ 16) on a
    second thread and stream: the dt sequence and the final state must be the bits of the same advance run alone."""
    import threading
    w = wl.config_3_cosmo(64, seed=31)
    hot = torch.from_numpy(wl.config_2_turbulence(64, seed=4).groups()).to(DEV)
    v_hot = gh.gamer_hydro_max_speed(hot)
    steps = 12

    def advance(out):
        st = torch.cuda.Stream()
        with torch.cuda.stream(st):
            d_U = torch.from_numpy(w.groups()).to(DEV)
            d_out = torch.empty((d_U.shape[0], 5, 16, 16, 16), dtype=torch.float32, device=DEV)
            dts = gh.gamer_hydro_advance(d_U, d_out, None, _grid(w.shape), steps, 0.4, pu.f32(w.dx),
                                         bc=[BC[b] for b in w.bc], limiter=w.limiter, stream=st)
            st.synchronize()
            out.append((dts, d_U.cpu().numpy()))

    alone = []
    advance(alone)
    for rep in range(2):
        both, seen, stop = [], [], threading.Event()

        def hammer():
            st = torch.cuda.Stream()
            while not stop.is_set() or len(seen) < 400:
                seen.append(gh.gamer_hydro_max_speed(hot, stream=st))

        t1, t2 = threading.Thread(target=advance, args=(both,)), threading.Thread(target=hammer)
        t2.start(); t1.start(); t1.join(); stop.set(); t2.join()
        assert len(seen) >= 400 and all(v == v_hot for v in seen)             # nor did the advance disturb the hammer
        assert both[0][0] == alone[0][0]                                      # same dt sequence, bit for bit
        assert np.array_equal(both[0][1], alone[0][1])


def test_generic_path_steps_of_growing_shapes_on_two_threads():
    """launch_generic used to read the scratch address outside the lock under which another thread may
    free and re-allocate it for a larger shape. Two host threads step generic shapes (N = 8 / ghost 2 and N = 12 /
    ghost 3: the second needs the larger scratch, and both start before it exists) on their own streams; every result
    must be the bits of the same call made alone."""
    import threading
    shapes = [(8, 2, 40), (12, 3, 24)]
    rng = np.random.default_rng(77)
    data = []
    for N, ghost, n in shapes:
        S = N + 2 * ghost
        U = np.empty((n, 5, S, S, S), dtype=np.float32)
        U[:, 0] = rng.uniform(0.5, 2.0, (n, S, S, S))
        U[:, 1:4] = rng.uniform(-0.3, 0.3, (n, 3, S, S, S)) * U[:, :1]
        U[:, 4] = rng.uniform(1.0, 2.0, (n, S, S, S)) / (G - 1.0) + 0.5 * (U[:, 1:4] ** 2).sum(axis=1) / U[:, 0]
        data.append(torch.from_numpy(U).to(DEV))
    dt, dx = pu.f32(2e-3), pu.f32(1.0 / 32)

    def step(k, st, out):
        N, ghost, n = shapes[k]
        with torch.cuda.stream(st):
            o = torch.full((n, 5, N, N, N), float("nan"), dtype=torch.float32, device=DEV)
            bf = torch.full((n, 6, 5, N, N), float("nan"), dtype=torch.float32, device=DEV)
            gh.gamer_hydro_step(data[k], o, bf, n, N, ghost, dt, dx, G, gh.MINMOD, stream=st)
            st.synchronize()
            out.append((o.cpu().numpy(), bf.cpu().numpy()))

    gh.gamer_hydro_free()                                       # start without any scratch: the first calls grow it
    conc = [[], []]

    def loop(k):
        st = torch.cuda.Stream()
        for _ in range(20):
            step(k, st, conc[k])

    th = [threading.Thread(target=loop, args=(k,)) for k in range(2)]
    for t in th:
        t.start()
    for t in th:
        t.join()
    for k in range(2):
        ref = []
        step(k, torch.cuda.Stream(), ref)
        assert np.isfinite(ref[0][0]).all() and np.isfinite(ref[0][1]).all()
        for o, bf in conc[k]:
            assert np.array_equal(o, ref[0][0]) and np.array_equal(bf, ref[0][1])
