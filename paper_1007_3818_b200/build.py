"""Builds the C-ABI shared library paper_1007_3818_b200/libgamer_hydro.so for sm_100a (in-tree, so that the
.so travels to the GPU box with the snapshot). nvcc cross-compiles without a GPU."""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libgamer_hydro.so")
SOURCES = ["gamer_hydro_api.cu"]
DEPS = ["gamer_hydro_api.cu", "hydro_fused.cuh", "hydro_f2.cuh", "hydro_duo.cuh", "hydro_zpair.cuh", "hydro_aux.cuh", "hydro_rtvd.cuh", "hydro_generic.cuh", "hydro_math.cuh",
        os.path.join("..", "..", "include", "gamer_hydro.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "-shared",
              "-Xcompiler", "-fPIC", "-Xptxas", "-v", "--expt-relaxed-constexpr"]


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(os.path.join(CSRC, d)) > t for d in DEPS) or os.path.getmtime(__file__) > t


def build(force: bool = False, verbose: bool = False) -> str:
    if force or needs_build():
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        tmp = LIB + ".tmp.%d" % os.getpid()
        cmd = [nvcc] + NVCC_FLAGS + ["-o", tmp] + [os.path.join(CSRC, s) for s in SOURCES]
        res = subprocess.run(cmd, cwd=CSRC, capture_output=True, text=True)
        if verbose or res.returncode != 0:
            print(res.stdout)
            print(res.stderr)
        res.check_returncode()
        os.replace(tmp, LIB)
        with open(os.path.join(HERE, "build_ptxas.log"), "w") as f:
            f.write(res.stderr)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
