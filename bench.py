#!/usr/bin/env python
"""bench.py — cell-updates/s of the fused MUSCL-Hancock + Roe step on B200, with roofline.

One "step" = one pass of the whole hot path (reconstruction, half-step prediction, Roe solver, full-step
update, boundary fluxes) over one batch of synthetic patch groups. At N = 1 the workload is
BASELINE.json:configs[3], the configuration the metric is quoted on: 32768 groups of 16^3 cells (+2 ghost
layers) cut from a seeded 512^3 cosmology-like baryonic field, fp32, gamma = 5/3, MinMod, one step per
launch. With N > 1 there is one rank per GPU (`python bench.py --gpus N` re-executes itself under
torch.distributed.run when it was not started by it); patch groups are independent, so the path shards with no
collective: `--scaling weak` (default) gives every rank the full 32768-group batch, `--scaling strong` splits the ONE
batch into contiguous group ranges (paper_1007_3818_b200/sharding.py). The field is generated once (rank 0) and
shared with the other ranks through a file in /dev/shm.

Contract: `python bench.py --gpus N --steps K --warmup W [--impl reference]` prints ONE JSON line on rank 0.
  value      whole-job cell-updates/s with inputs resident in HBM (CUDA events, max over ranks)
  e2e        same metric through the C-ABI host-buffer call gamer_hydro_step_host (pinned host memory,
             H2D + kernels + D2H inside the timed region)
  roofline   ALU-bound: counted algorithmic FLOPs (the oracle's CountingReal tally) / time
             against 148 SM x 128 lanes x 2 x 1.965 GHz; the HBM side is reported next to it
  cpu_baseline  the fp64 oracle as it stands, on this box's host cores, on a bounded sample of the same
             workload (rank 0, N = 1 only); the same sample doubles as a parity spot-check
`--impl reference` times the oracle alone (this tier's reference arm).
"""
import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "cell-updates/s (fp32 MUSCL-Hancock+Roe step, 16^3 patch groups with 2-cell ghost shell)"
UNIT = "cell-updates/s"
N, GHOST = 16, 2
# algorithmic FLOPs per cell-update: oracle CountingReal tally on an all-slopes-active field (
# tests/test_oracle_pins.py::test_flop_tally_band re-derives it). Hand count of SURVEY.md App. D: 925 / 966.
FLOPS_PER_CELL = {0: 1033.94, 1: 1095.81}
FLOPS_PER_CELL_HAND = {0: 925.0, 1: 966.0}
BYTES_PER_CELL = 66.5625           # (5*20^3 + 5*16^3 + 30*16^2) * 4 B / 16^3
# relaxing-TVD step: the oracle text run with the counting scalar of oracle/counting_real.hpp
# (oracle.rtvd_oracle.count_flops: 1200.3 / 1200.2 for the two sweep orders; 1092 lines of 22 cells per group), held to
# a hand count by tests/test_rtvd_oracle_pins.py. Rounds 1-2 printed 1279, a hand count that was 6.6 % too high.
RTVD_FLOPS_PER_CELL = 1200.0
RTVD_BYTES_PER_CELL = (5 * 22 ** 3 + 5 * 16 ** 3) * 4 / 16 ** 3      # 72.0
SM_COUNT, LANES, SM_MAX_GHZ = 148, 128, 1.965
ALU_PEAK_TFLOPS = SM_COUNT * LANES * 2 * SM_MAX_GHZ / 1e3     # 74.45
FP64_PEAK_TFLOPS = SM_COUNT * 64 * 2 * SM_MAX_GHZ / 1e3        # 37.22
ISSUE_COST_PER_CELL = 960.0     # scheduler clocks per cell-update the MinMod z-pair kernel's instruction mix costs (profiles/r2b_README.md)


def measured_hbm_peak():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index, period=0.02):
        super().__init__(daemon=True)
        self.index, self.period = index, period
        self.samples, self.reasons, self.stop_flag = [], set(), False
        self.max_mhz = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def run(self):
        if self.nv is None:
            return
        nv = self.nv
        names = {nv.nvmlClocksThrottleReasonSwPowerCap: "sw_power_cap",
                 nv.nvmlClocksThrottleReasonHwSlowdown: "hw_slowdown",
                 nv.nvmlClocksThrottleReasonHwThermalSlowdown: "hw_thermal_slowdown",
                 nv.nvmlClocksThrottleReasonSwThermalSlowdown: "sw_thermal_slowdown",
                 nv.nvmlClocksThrottleReasonHwPowerBrakeSlowdown: "hw_power_brake"}
        while not self.stop_flag:
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, name in names.items():
                    if r & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            time.sleep(self.period)

    def result(self):
        self.stop_flag = True
        if self.is_alive():
            self.join()
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": ["nvml unavailable"]}
        return {"sm_mhz": float(np.median(self.samples)), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.samples)}


def make_workload(n_box, seed):
    from harness import workloads as wl
    t0 = time.time()
    w = wl.config_3_cosmo(n_box, seed=seed)
    groups = w.groups(np.float32)
    dt = w.dt()
    dx = float(np.float32(w.dx))
    return w, groups, dt, dx, time.time() - t0


def run_reference(args, rank, world):
    """This tier's reference arm: the fp64 oracle alone, on the host cores, on a bounded sample per step."""
    if rank != 0:
        return
    from oracle import mhm_oracle as O
    w, groups, dt, dx, _ = make_workload(128, args.seed)     # 512 groups of the same recipe: a bounded sample
    sample = groups[: args.ref_groups]
    for _ in range(args.warmup):
        O.step_groups(sample, N, GHOST, dt, dx, w.gamma, w.limiter, want_guard=False)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        r = O.step_groups(sample, N, GHOST, dt, dx, w.gamma, w.limiter, want_guard=False)
    t = time.perf_counter() - t0
    cells = sample.shape[0] * N ** 3 * args.steps
    val = cells / t
    desc = "%d groups of the cfg3 recipe (128^3 box) per step, all host cores" % sample.shape[0]
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * t / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "cfg3_cosmo (BASELINE.json:configs[3]) bounded sample: " + desc,
                   "limiter": "minmod", "gamma": w.gamma},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": r.threads, "kind": "oracle", "sample": desc},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


def maybe_respawn(args):
    """`python bench.py --gpus N` with N > 1 and no torchrun environment: start N ranks of this script under
    torch.distributed.run on this node (one GPU each) and exit with their status."""
    if args.gpus <= 1 or "WORLD_SIZE" in os.environ:
        return
    import socket
    import subprocess
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus),
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    raise SystemExit(subprocess.call(cmd))


def shared_workload(args, rank, world, barrier):
    """The cfg3 field, generated ONCE (rank 0) and shared with the other ranks of the node through /dev/shm."""
    if world == 1:
        return make_workload(args.box, args.seed)
    from harness import workloads as wl
    tag = "gamer_bench_%s_%d_%d" % (os.environ.get("MASTER_PORT", "0"), args.box, args.seed)
    base = os.path.join("/dev/shm" if os.path.isdir("/dev/shm") else "/tmp", tag)
    t0 = time.time()
    if rank == 0:
        w, groups, dt, dx, _ = make_workload(args.box, args.seed)
        np.save(base + ".npy", groups)
        with open(base + ".json", "w") as f:
            json.dump({"dt": dt, "dx": dx}, f)
    barrier()
    if rank != 0:
        w = wl.Workload("cfg3_cosmo_%d" % args.box, None, 1.0 / args.box, ("periodic",) * 3, 0, 0.5, 1)
        groups = np.load(base + ".npy", mmap_mode="r")
        with open(base + ".json") as f:
            meta = json.load(f)
        dt, dx = meta["dt"], meta["dx"]
    barrier()
    if rank == 0:
        for ext in (".npy", ".json"):
            try:
                os.remove(base + ext)
            except OSError:
                pass
    return w, groups, dt, dx, time.time() - t0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--box", type=int, default=512, help="global box edge; 512 -> 32768 groups (headline)")
    ap.add_argument("--seed", type=int, default=3)
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"],
                    help="N > 1: weak = the full batch on every rank; strong = the one batch split by sharding.shard_range")
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--cpu-groups", type=int, default=4096,
                    help="groups in the oracle sample (cpu_baseline): 16.8 M cell-updates, about 15 core-seconds")
    ap.add_argument("--ref-groups", type=int, default=512,
                    help="groups per step of the --impl reference arm (its 128^3 box holds 512)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-multistep", action="store_true")
    ap.add_argument("--no-cuda", action="store_true",
                    help="launcher self-test (CPU, gloo): everything up to, not including, the first CUDA call")
    ap.add_argument("--path", default="auto", choices=["auto", "generic", "fused", "fused_scalar", "fused_duo"],
                    help="kernel path forced through gamer_hydro_set_path (default: the library's choice)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "ours":
        maybe_respawn(args)

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.impl == "reference":
        run_reference(args, rank, world)
        return

    import torch
    import torch.distributed as dist
    from paper_1007_3818_b200 import sharding

    if args.no_cuda:
        # the N > 1 plumbing without a GPU: rendezvous, one field for all ranks, the partition, the timing reduction
        if world > 1:
            dist.init_process_group("gloo")
        cpu_barrier = (lambda: dist.barrier()) if world > 1 else (lambda: None)
        w, groups, dt, dx, gen_s = shared_workload(args, rank, world, cpu_barrier)
        a, b = sharding.shard_range(groups.shape[0], rank, world) if args.scaling == "strong" else (0, groups.shape[0])
        mine = np.ascontiguousarray(groups[a:b])
        t = sharding.max_over_ranks(1.0 + rank)
        counts = torch.tensor([b - a], dtype=torch.int64)
        if world > 1:
            dist.all_reduce(counts)
        if rank == 0:
            print(json.dumps({"launcher_self_test": True, "n_gpus": world, "scaling": args.scaling,
                              "groups_total": int(counts.item()), "groups_rank0": int(mine.shape[0]),
                              "max_over_ranks": t, "checksum_rank0": float(np.asarray(mine, dtype=np.float64).sum())}))
        if world > 1:
            dist.destroy_process_group()
        return

    import paper_1007_3818_b200 as gh

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    w, all_groups, dt, dx, gen_s = shared_workload(args, rank, world, barrier)
    g0, g1 = sharding.shard_range(all_groups.shape[0], rank, world) if args.scaling == "strong" else (0, all_groups.shape[0])
    groups = np.ascontiguousarray(all_groups[g0:g1])
    G = groups.shape[0]
    cells = G * N ** 3
    gh.gamer_hydro_alloc(G, N, GHOST, 4, local_rank)
    gh.gamer_hydro_set_path({"auto": 0, "generic": 1, "fused": 2, "fused_scalar": 3, "fused_duo": 4}[args.path])
    h_in = torch.from_numpy(groups)
    d_in = h_in.to(dev)
    d_out = torch.empty((G, 5, N, N, N), dtype=torch.float32, device=dev)
    d_bf = torch.empty((G, 6, 5, N, N), dtype=torch.float32, device=dev)
    stream = torch.cuda.current_stream()

    def step():
        gh.gamer_hydro_step(d_in, d_out, d_bf, G, N, GHOST, dt, dx, w.gamma, w.limiter, stream=stream)

    for _ in range(args.warmup):
        step()
    barrier()
    gh.gamer_hydro_status()                                   # reset the diagnostics counters
    sampler = ClockSampler(local_rank)
    sampler.start()
    evs = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
    launches0 = gh.gamer_hydro_launch_count()
    barrier()
    evs[0].record(stream)
    for s in range(args.steps):
        step()
        evs[s + 1].record(stream)
    barrier()
    clocks = sampler.result()
    launches = gh.gamer_hydro_launch_count() - launches0
    total_ms = evs[0].elapsed_time(evs[-1])
    per_step = [evs[s].elapsed_time(evs[s + 1]) for s in range(args.steps)]
    guard_cells, nonpos = gh.gamer_hydro_status()
    total_ms_max = sharding.max_over_ranks(total_ms, device=dev)          # the slowest rank sets the job's time
    cells_all = cells
    if world > 1:
        ct = torch.tensor([cells], dtype=torch.int64, device=dev)
        dist.all_reduce(ct)
        cells_all = int(ct.item())
    value = cells_all * args.steps / (total_ms_max * 1e-3)                # == sharding.aggregate_throughput for equal shards

    # ---- e2e: host buffers through the C ABI, copies inside the timed region
    e2e = None
    if not args.no_e2e:
        hp_in = h_in.pin_memory()
        hp_out = torch.empty((G, 5, N, N, N), dtype=torch.float32).pin_memory()
        hp_bf = torch.empty((G, 6, 5, N, N), dtype=torch.float32).pin_memory()

        def e2e_step():
            gh.gamer_hydro_step_host(hp_in, hp_out, hp_bf, G, N, GHOST, dt, dx, w.gamma, w.limiter, chunk_groups=0)

        e2e_step()
        barrier()
        t0 = time.perf_counter()
        for _ in range(args.e2e_steps):
            e2e_step()
        barrier()
        te = sharding.max_over_ranks(time.perf_counter() - t0, device=dev)
        h2d_b, d2h_b = int(hp_in.numel() * 4), int((hp_out.numel() + hp_bf.numel()) * 4)
        # the host link's own speed, measured in the same run: one pinned H2D copy of the input, one D2H of the output
        c0, c1, c2 = (torch.cuda.Event(enable_timing=True) for _ in range(3))
        d_in.copy_(hp_in, non_blocking=True)
        barrier()
        c0.record(stream)
        d_in.copy_(hp_in, non_blocking=True)
        c1.record(stream)
        hp_out.copy_(d_out, non_blocking=True)
        c2.record(stream)
        barrier()
        h2d_peak = h2d_b / (c0.elapsed_time(c1) * 1e-3) / 1e9
        d2h_peak = hp_out.numel() * 4 / (c1.elapsed_time(c2) * 1e-3) / 1e9
        t_step = te / args.e2e_steps
        # H2D and D2H run on different copy engines and overlap: the link-bound time of a step is the longer of the two
        t_link = max(h2d_b / (h2d_peak * 1e9), d2h_b / (d2h_peak * 1e9))
        e2e = {"value": cells_all * args.e2e_steps / te, "unit": UNIT,
               "h2d_bytes_per_step": h2d_b, "d2h_bytes_per_step": d2h_b, "steps": args.e2e_steps,
               "api": "gamer_hydro_step_host (pinned host buffers, chunked 3-stream overlap)",
               "h2d_gbs_achieved": h2d_b / t_step / 1e9, "d2h_gbs_achieved": d2h_b / t_step / 1e9,
               "h2d_gbs_pinned_copy_alone": h2d_peak, "d2h_gbs_pinned_copy_alone": d2h_peak,
               "frac_of_link_bound_time": t_link / t_step}
        e2e["matches_device_path_bitwise"] = bool(torch.equal(hp_out, d_out.cpu()))
        del hp_in, hp_out, hp_bf

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant (only) kernel of the step
    ms_launch = total_ms / args.steps                         # one launch per step on this rank
    flops = FLOPS_PER_CELL[w.limiter] * cells
    achieved_tf = flops / (ms_launch * 1e-3) / 1e12
    hbm_peak, hbm_src = measured_hbm_peak()
    hbm_gbs = BYTES_PER_CELL * cells / (ms_launch * 1e-3) / 1e9
    traffic, traffic_src = None, None
    try:
        with open(os.path.join(ROOT, "profiles", "r3_traffic_bytes_per_launch.txt")) as f:
            tj = json.load(f)
            if tj.get("n_groups") == G and args.path in ("auto", "fused"):
                traffic = tj["dram_bytes_read_plus_write"]
                traffic_src = "ncu --set full capture, profiles/r3_traffic_bytes_per_launch.txt (commit %s)" % tj.get("commit")
    except Exception:
        pass
    roofline = {"bound": "alu", "achieved": achieved_tf, "peak": ALU_PEAK_TFLOPS, "unit": "TFLOP/s",
                "frac": achieved_tf / ALU_PEAK_TFLOPS, "traffic": traffic, "traffic_source": traffic_src,
                "kernel": {"auto": "gh::zpair_kernel<MinMod>", "fused": "gh::zpair_kernel<MinMod>",
                           "fused_scalar": "gh::fused_kernel<float, MinMod, fast>",
                           "fused_duo": "gh::duo_kernel<MinMod>",
                           "generic": "gh::predict_kernel + flux_kernel + update_kernel"}[args.path],
                "flops_per_cell_update": FLOPS_PER_CELL[w.limiter],
                "flops_source": "oracle CountingReal tally (DESIGN.md section 6); SURVEY.md App. D hand count: %g"
                                % FLOPS_PER_CELL_HAND[w.limiter],
                "frac_with_hand_count": FLOPS_PER_CELL_HAND[w.limiter] * cells / (ms_launch * 1e-3) / 1e12 / ALU_PEAK_TFLOPS,
                "target_frac": 0.60, "target_met": bool(achieved_tf / ALU_PEAK_TFLOPS >= 0.60),
                "peak_derivation": "148 SM x 128 FP32 lanes x 2 FLOP x 1.965 GHz (sm_max_mhz of MEASURED_PEAKS.json)",
                "ms_per_launch": ms_launch,
                "hbm": {"algorithmic_bytes_per_launch": BYTES_PER_CELL * cells, "achieved_gbs": hbm_gbs,
                        "peak_gbs": hbm_peak, "peak_source": hbm_src, "frac": hbm_gbs / hbm_peak},
                "frac_of_binding_roofline_time": max(flops / (ALU_PEAK_TFLOPS * 1e12),
                                                     BYTES_PER_CELL * cells / (hbm_peak * 1e9)) / (ms_launch * 1e-3)}
    if args.path in ("auto", "fused") and w.limiter == 0:
        # what the step costs the warp schedulers (explanatory, not a roofline): scheduler clocks per cell-update of this
        # run against the issue cost of the kernel's executed instruction mix (profiles/r2b_README.md: packed f32x2 = 2
        # clocks, 3 with three distinct source pairs; measured by harness/issue_microbench.py)
        sched_clocks = ms_launch * 1e-3 * SM_MAX_GHZ * 1e9 * SM_COUNT * 4 * 32 / cells
        roofline["issue_model"] = {"kind": "MODEL, not a counter: executed instruction mix (profiles/r3_zpair_opcode_mix.csv) "
                                           "x per-opcode issue cost (harness/issue_microbench.py); ncu's own counter is "
                                           "smsp__issue_active in profiles/r3_zpair_kernel_ncu_full.csv",
                                   "scheduler_clocks_per_cell_update": sched_clocks,
                                   "modelled_issue_cost_of_instruction_mix": ISSUE_COST_PER_CELL,
                                   "modelled_frac_of_issue_bound": ISSUE_COST_PER_CELL / sched_clocks,
                                   "clocks_at_target_frac": FLOPS_PER_CELL[0] / (2 * 0.60),
                                   "source": "profiles/r2b_README.md, harness/issue_microbench.py"}

    # ---- cpu_baseline: the oracle on a bounded sample of the same workload (+ parity spot-check)
    cpu = None
    if not args.no_cpu_baseline and world == 1:
        from oracle import mhm_oracle as O
        from harness import metrics
        rng = np.random.default_rng(12345)
        rho_max = groups[:, 0, 2:-2, 2:-2, 2:-2].reshape(G, -1).max(axis=1)
        pick = set(int(i) for i in rng.choice(G, size=min(args.cpu_groups, G) - 2, replace=False))
        pick.update([int(np.argmax(rho_max)), int(np.argmin(rho_max))])
        idx = np.array(sorted(pick))
        sample = np.ascontiguousarray(groups[idx])
        t0 = time.perf_counter()
        r = O.step_groups(sample, N, GHOST, dt, dx, w.gamma, w.limiter)
        tc = time.perf_counter() - t0
        n1 = min(256, len(idx))                               # one thread: a smaller sample of the same groups
        t0 = time.perf_counter()
        O.step_groups(sample[:n1], N, GHOST, dt, dx, w.gamma, w.limiter, n_threads=1)
        t1 = time.perf_counter() - t0
        gout = d_out[torch.from_numpy(idx).to(dev)].cpu().numpy()
        sus = metrics.suspect_mask(r.margin)
        err = metrics.max_rel_err(gout, r.U_out, w.gamma, mask=np.broadcast_to(~sus[:, None], r.U_out.shape))
        desc = "%d of the %d groups (seeded random + the groups holding max/min density), one step" % (len(idx), G)
        cpu = {"value": len(idx) * N ** 3 / tc, "unit": UNIT, "cores": r.threads, "kind": "oracle", "sample": desc,
               "seconds": tc, "one_thread": {"value": n1 * N ** 3 / t1, "unit": UNIT, "cores": 1, "seconds": t1,
                                             "sample": "the first %d groups of the same sample" % n1},
               "parity_max_rel_err_on_sample": err, "parity_tolerance": 1e-4,
               "parity_excluded_fraction": float(sus.mean()), "oracle_guard_cells_on_sample": r.guard_cells}

    # ---- device-resident multi-step run on the same grid: signal-speed maximum + step + ghost
    # refill per step, one 4-byte D2H read per step; reported beside the headline, not part of it
    multistep = None
    if not args.no_multistep and world == 1:
        gpa = args.box // N
        d_state = d_in.clone()
        gh.gamer_hydro_advance(d_state, d_out, d_bf, (gpa, gpa, gpa), 2, 0.5, dx, gamma=w.gamma, limiter=w.limiter)
        torch.cuda.synchronize()
        nms = 6
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        ms_dts = gh.gamer_hydro_advance(d_state, d_out, d_bf, (gpa, gpa, gpa), nms, 0.5, dx, gamma=w.gamma,
                                        limiter=w.limiter)
        e1.record(stream)
        torch.cuda.synchronize()
        ms_ms = e0.elapsed_time(e1) / nms
        multistep = {"value": cells / (ms_ms * 1e-3), "unit": UNIT, "steps": nms, "ms_per_step": ms_ms,
                     "api": "gamer_hydro_advance on the periodic grid (per step: the step kernel, the ghost-refill kernel "
                            "that also accumulates the next signal-speed maximum, one 4-byte D2H read)",
                     "dt_first": ms_dts[0], "dt_last": ms_dts[-1]}
        del d_state

    # ---- second workload: the relaxing-TVD step on a 256^3 box of the same recipe with 3 ghost
    # cells (4096 groups), beside the headline, with its own roofline
    rtvd = None
    if not args.no_multistep and world == 1:
        from harness import workloads as wl
        w2 = wl.config_3_cosmo(min(args.box, 256), seed=args.seed)
        g3 = torch.from_numpy(wl.cut_groups(w2.U, w2.bc, ghost=3)).to(dev)
        n3 = g3.shape[0]
        o3 = torch.empty((n3, 5, N, N, N), dtype=torch.float32, device=dev)
        dt3, dx3 = float(np.float32(w2.dt())), float(np.float32(w2.dx))
        for s in range(3):
            gh.gamer_rtvd_step(g3, o3, n3, N, 3, dt3, dx3, w2.gamma, s % 2, stream=stream)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record(stream)
        for s in range(10):
            gh.gamer_rtvd_step(g3, o3, n3, N, 3, dt3, dx3, w2.gamma, s % 2, stream=stream)
        e1.record(stream)
        torch.cuda.synchronize()
        ms3 = e0.elapsed_time(e1) / 10
        c3 = n3 * N ** 3
        # parity spot-check on the input just timed (as the headline has): 64 groups spread over the batch, one step in
        # either sweep order against the fp64 oracle (all 4096 groups: tests/test_gpu_rtvd.py)
        rtvd_parity = None
        if not args.no_cpu_baseline:
            from oracle import rtvd_oracle as RO
            from harness import metrics as hm
            pick = np.arange(0, n3, max(1, n3 // 64))[:64]
            sub = g3[torch.from_numpy(pick).to(dev)].contiguous()
            rtvd_parity = 0.0
            for sw in (0, 1):
                o_s = torch.empty((len(pick), 5, N, N, N), dtype=torch.float32, device=dev)
                gh.gamer_rtvd_step(sub, o_s, len(pick), N, 3, dt3, dx3, w2.gamma, sw, stream=stream)
                torch.cuda.synchronize()
                ref_s, _ = RO.step_groups(sub.cpu().numpy(), N, dt3, dx3, w2.gamma, sw)
                rtvd_parity = max(rtvd_parity, float(hm.max_rel_err(o_s.cpu().numpy(), ref_s, w2.gamma)))
        rtvd = {"value": c3 / (ms3 * 1e-3), "unit": UNIT, "ms_per_step": ms3, "groups": n3, "ghost": 3,
                "api": "gamer_rtvd_step (x,y,z / z,y,x sweeps alternating)", "kernel": "gh::rtvd_kernel",
                "parity_max_rel_err_on_sample": rtvd_parity, "parity_tolerance": 1e-4,
                "parity_sample": "64 of the timed groups, both sweep orders, vs oracle/rtvd_oracle.hpp",
                "roofline": {"bound": "alu", "flops_per_cell_update": RTVD_FLOPS_PER_CELL,
                             "achieved": RTVD_FLOPS_PER_CELL * c3 / (ms3 * 1e-3) / 1e12, "peak": ALU_PEAK_TFLOPS,
                             "unit": "TFLOP/s", "frac": RTVD_FLOPS_PER_CELL * c3 / (ms3 * 1e-3) / 1e12 / ALU_PEAK_TFLOPS,
                             "hbm_bytes_per_cell_update": RTVD_BYTES_PER_CELL,
                             "hbm_frac": RTVD_BYTES_PER_CELL * c3 / (ms3 * 1e-3) / 1e9 / hbm_peak}}
        del g3, o3

    # ---- the fp64 entry (the 1e-11 parity path) on the 256^3 box of the same recipe, with its own roofline
    f64 = None
    if not args.no_multistep and world == 1:
        from harness import workloads as wl
        w4 = wl.config_3_cosmo(min(args.box, 256), seed=args.seed)
        g4 = torch.from_numpy(wl.cut_groups(w4.U, w4.bc, ghost=2).astype(np.float64)).to(dev)
        n4 = g4.shape[0]
        o4 = torch.empty((n4, 5, N, N, N), dtype=torch.float64, device=dev)
        b4 = torch.empty((n4, 6, 5, N, N), dtype=torch.float64, device=dev)
        dt4, dx4 = float(w4.dt()), float(w4.dx)
        for s in range(3):
            gh.gamer_hydro_step_f64(g4, o4, b4, n4, N, 2, dt4, dx4, w4.gamma, 0, stream=stream)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record(stream)
        for s in range(10):
            gh.gamer_hydro_step_f64(g4, o4, b4, n4, N, 2, dt4, dx4, w4.gamma, 0, stream=stream)
        e1.record(stream)
        torch.cuda.synchronize()
        ms4 = e0.elapsed_time(e1) / 10
        c4 = n4 * N ** 3
        tf4 = FLOPS_PER_CELL[0] * c4 / (ms4 * 1e-3) / 1e12
        f64 = {"value": c4 / (ms4 * 1e-3), "unit": UNIT, "ms_per_step": ms4, "groups": n4, "dtype": "f64",
               "api": "gamer_hydro_step_f64", "kernel": "gh::fused_kernel<double, MinMod>",
               "roofline": {"bound": "alu (fp64)", "flops_per_cell_update": FLOPS_PER_CELL[0], "achieved": tf4,
                            "peak": FP64_PEAK_TFLOPS, "unit": "TFLOP/s", "frac": tf4 / FP64_PEAK_TFLOPS,
                            "peak_derivation": "148 SM x 64 FP64 lanes x 2 FLOP x 1.965 GHz (DFMA rate measured by "
                                               "harness/issue_microbench.py: 2 clocks per warp instruction and scheduler)",
                            "hbm_frac": 2 * BYTES_PER_CELL * c4 / (ms4 * 1e-3) / 1e9 / hbm_peak}}
        del g4, o4, b4

    out = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
           "warmup": args.warmup, "ms_per_step": total_ms_max / args.steps, "higher_is_better": True,
           "scaling": args.scaling if world > 1 else "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
           "config": {"workload": "cfg3_cosmo_%d (BASELINE.json:configs[3]): %d patch groups/GPU, 16^3+2 ghost, "
                                  "5 vars, gamma=5/3, MinMod, 1 step per launch" % (args.box, G),
                      "groups_per_gpu": G, "cells_per_gpu": cells, "cells_all_gpus": cells_all, "seed": args.seed,
                      "l2": "inputs (%.2f GB/step) far larger than the 126 MB L2; no flush needed" %
                            (h_in.numel() * 4 / 1e9),
                      "parallelism": "groups sharded across ranks (%s), no collective" %
                                     ("the one batch split into contiguous ranges" if args.scaling == "strong" and world > 1
                                      else "the full batch on every rank"),
                      "generation_seconds": gen_s, "dt": dt, "dx": dx, "kernel_path": args.path},
           "roofline": roofline, "cpu_baseline": cpu, "e2e": e2e, "multistep": multistep, "rtvd": rtvd, "f64": f64,
           "gpu_launches": int(launches),
           "clocks": clocks, "ms_per_step_min": min(per_step), "ms_per_step_median": float(np.median(per_step)),
           "guard_cells_per_step": guard_cells / args.steps, "nonpositive_out_per_step": nonpos / args.steps,
           "context_paper": {"gpu_vs_cpu_solver_speedup": 55.0, "overall_speedup_8800GTX": 19.2,
                             "overall_speedup_T10_rtvd": 16.5, "source": "PAPER.md:27,29,13 (other hardware)"}}
    # the contract's keys keep their types (a local variable once shadowed the clocks record)
    assert isinstance(out["clocks"], dict) and isinstance(out["roofline"], dict) and isinstance(out["config"], dict)
    assert isinstance(out["gpu_launches"], int) and out["gpu_launches"] > 0
    print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
