"""CPU-side checks (-m "not gpu") of the boundary: libgamer_hydro.so builds for sm_100a, loads without a GPU and
exports every function include/gamer_hydro.h declares; argument validation that needs no device; the product
path has no CPU fallback (compute entries fail loudly here); nothing in the product imports the oracle."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_functions():
    src = open(os.path.join(ROOT, "include", "gamer_hydro.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(gamer_(?:hydro|rtvd)_[a-z0-9_]+)\s*\(", src)))


def test_header_declares_the_north_star_entry_points():
    names = declared_functions()
    assert "gamer_hydro_alloc" in names and "gamer_hydro_step" in names
    src = open(os.path.join(ROOT, "include", "gamer_hydro.h")).read()
    sig = re.sub(r"\s+", " ", src)
    assert ("int gamer_hydro_step(const float* U_in_with_ghosts, float* U_out, float* boundary_fluxes, int n_groups, "
            "int N, int ghost, float dt, float dx, float gamma, int limiter, cudaStream_t stream);") in sig


def test_library_builds_loads_and_exports_every_declared_symbol():
    from paper_1007_3818_b200 import binding, build
    path = build.build()
    L = C.CDLL(path)
    for name in declared_functions():
        assert hasattr(L, name), name
    assert sorted(binding.EXPORTS) == declared_functions()
    # the binding mirrors the header one to one
    import paper_1007_3818_b200 as gh
    for name in declared_functions():
        assert callable(getattr(gh, name)), name


def test_sass_contains_tma_and_mbarrier_instructions():
    """Evidence that the fused kernel is the sm_100a TMA path (B200_PROFILING.md: UTMALDG = cp.async.bulk.tensor)."""
    import shutil
    import subprocess
    from paper_1007_3818_b200 import build
    if shutil.which("cuobjdump") is None and not os.path.exists("/usr/local/cuda/bin/cuobjdump"):
        pytest.skip("cuobjdump not available")
    exe = shutil.which("cuobjdump") or "/usr/local/cuda/bin/cuobjdump"
    sass = subprocess.run([exe, "-sass", build.build()], capture_output=True, text=True, check=True).stdout
    assert "sm_100a" in sass and "UTMALDG" in sass and "SYNCS" in sass


def test_strerror_and_argument_validation_without_a_device():
    import paper_1007_3818_b200 as gh
    assert gh.gamer_hydro_strerror(0) == "success"
    assert "invalid" in gh.gamer_hydro_strerror(1)
    assert "64" in gh.gamer_hydro_strerror(6) and "unknown" in gh.gamer_hydro_strerror(7)     # GAMER_HYDRO_BUSY; no code 7
    L = gh.binding.lib()
    # validation happens before any CUDA call, so these return INVALID_ARG (1) even on a box with no GPU
    assert L.gamer_hydro_step(None, None, None, -1, 16, 2, 1e-3, 1e-2, 5 / 3, 0, None) == 1
    assert L.gamer_hydro_step(None, None, None, 4, 16, 1, 1e-3, 1e-2, 5 / 3, 0, None) == 1      # ghost < 2
    assert L.gamer_hydro_step(None, None, None, 4, 16, 2, 0.0, 1e-2, 5 / 3, 0, None) == 1       # dt <= 0
    assert L.gamer_hydro_step(None, None, None, 4, 16, 2, 1e-3, 1e-2, 1.0, 0, None) == 1        # gamma <= 1
    assert L.gamer_hydro_step(None, None, None, 4, 16, 2, 1e-3, 1e-2, 5 / 3, 9, None) == 1      # limiter
    assert L.gamer_hydro_step(None, None, None, 4, 16, 2, 1e-3, 1e-2, 5 / 3, 0, None) == 1      # null buffers
    assert L.gamer_hydro_step(None, None, None, 0, 16, 2, 1e-3, 1e-2, 5 / 3, 0, None) == 0      # empty batch: no-op
    assert L.gamer_hydro_alloc(8, 16, 2, 3, 0) == 1                                             # bytes_per_real
    import ctypes
    vmax = ctypes.c_double(-1.0)
    assert L.gamer_hydro_max_speed(None, 4, 4, 16, 2, 5 / 3, ctypes.byref(vmax), None) == 1     # null array
    assert L.gamer_hydro_max_speed(None, 2, 4, 16, 2, 5 / 3, ctypes.byref(vmax), None) == 1     # bytes_per_real
    assert L.gamer_hydro_fill_ghosts(None, None, 4, 1, 1, 1, 16, 2, 0, 0, 0, None) == 1         # null arrays
    assert L.gamer_hydro_advance(None, None, None, 1, 1, 1, 16, 2, 0, 0, 0, 1, 0.5, 1.0, 5 / 3, 0, None, None) == 1


def test_no_cpu_fallback_without_a_gpu():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    import paper_1007_3818_b200 as gh
    with pytest.raises(gh.GamerHydroError):
        gh.gamer_hydro_alloc(8, 16, 2, 4, 0)
    x = torch.ones((1, 5, 20, 20, 20))
    out = torch.zeros((1, 5, 16, 16, 16))
    with pytest.raises(gh.GamerHydroError):
        gh.gamer_hydro_step(x, out, None, 1, 16, 2, 1e-3, 1e-2)          # CPU tensors are refused
    with pytest.raises(gh.GamerHydroError):
        gh.gamer_hydro_step_host(x, out, None, 1, 16, 2, 1e-3, 1e-2)     # no device: CUDA error surfaces


def test_product_never_imports_the_oracle_and_nothing_reads_work_dirs():
    pkg = os.path.join(ROOT, "paper_1007_3818_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                s = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+\S*oracle|#include\s+\S*oracle", s, flags=re.M), f
                assert "_work/" not in s and "/root/reference" not in s, f
    for f in ("bench.py", "__graft_entry__.py"):
        s = open(os.path.join(ROOT, f)).read()
        assert "/root/reference" not in s and "_work/" not in s


def test_workloads_module_is_arithmetic_free_of_both_sides():
    s = open(os.path.join(ROOT, "harness", "workloads.py")).read()
    assert not re.search(r"^\s*(from|import)\s+\S*(torch|binding|oracle)", s, flags=re.M)
    from harness import workloads as wl
    g = wl.random_groups(2, seed=1)
    assert g.shape == (2, 5, 20, 20, 20) and g.dtype == np.float32
    assert np.array_equal(g, wl.random_groups(2, seed=1))          # reproducible from the seed alone
    w = wl.config_0_sod3d()
    assert w.n_groups == 8 and w.groups().shape == (8, 5, 20, 20, 20)
    box = wl.assemble_box(w.groups()[:, :, 2:-2, 2:-2, 2:-2], w.shape)
    assert np.array_equal(box, w.U)


def test_issue_microbenchmark_generates_and_compiles_for_sm100a(tmp_path):
    """harness/issue_microbench.py (the evidence behind DESIGN.md section 6's issue-cost model): the generated source
    compiles for sm_100a and every timed loop still holds the instruction it is named after."""
    import shutil
    import subprocess
    from harness import issue_microbench as mb
    nvcc = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(nvcc):
        pytest.skip("nvcc not available")
    cu, exe = tmp_path / "mb.cu", tmp_path / "mb"
    cu.write_text(mb.generate())
    subprocess.run([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-o", str(exe), str(cu)], check=True)
    mix = mb.sass_mix(str(exe))
    lines = {l[:40].strip(): l[40:] for l in mix.split("\n")}
    assert "FFMA2" in lines["FFMA2 x*y+z (3 pairs)"] and "FADD2" in lines["FADD2"] and "DFMA" in lines["DFMA (fp64)"]
    assert "MUFU" in lines["4 FADD2 + MUFU.EX2"] and "LDS" in lines["4 FADD2 + LDS.64 (used)"]
