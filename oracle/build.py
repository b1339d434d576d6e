"""oracle/build.py — compiles the fp64 CPU oracle into oracle/libmhm_oracle.so (TEST INFRASTRUCTURE).

Flags follow SURVEY.md §7: -O2, floating-point contraction off (no FMA fusion, so the text of
mhm_oracle.hpp is what runs), OpenMP over patch groups. Called by __graft_entry__.build() and, on
demand, by oracle/mhm_oracle.py when the library is missing or older than its sources.
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SOURCES = ["mhm_oracle_capi.cpp", "mhm_oracle.hpp", "counting_real.hpp"]
LIB = os.path.join(HERE, "libmhm_oracle.so")


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(os.path.join(HERE, s)) > t for s in SOURCES)


def build(force: bool = False) -> str:
    if force or needs_build():
        tmp = LIB + ".tmp.%d" % os.getpid()
        cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC", "-Wall",
               "-o", tmp, os.path.join(HERE, "mhm_oracle_capi.cpp")]
        subprocess.run(cmd, check=True, cwd=HERE)
        os.replace(tmp, LIB)
    return LIB


RTVD_SOURCES = ["rtvd_oracle_capi.cpp", "rtvd_oracle.hpp", "counting_real.hpp"]
RTVD_LIB = os.path.join(HERE, "librtvd_oracle.so")


def build_rtvd(force: bool = False) -> str:
    """The relaxing-TVD oracle, same flags, its own library."""
    stale = not os.path.exists(RTVD_LIB) or any(os.path.getmtime(os.path.join(HERE, s)) > os.path.getmtime(RTVD_LIB)
                                                for s in RTVD_SOURCES)
    if force or stale:
        tmp = RTVD_LIB + ".tmp.%d" % os.getpid()
        cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC", "-Wall",
               "-o", tmp, os.path.join(HERE, "rtvd_oracle_capi.cpp")]
        subprocess.run(cmd, check=True, cwd=HERE)
        os.replace(tmp, RTVD_LIB)
    return RTVD_LIB


if __name__ == "__main__":
    print(build_rtvd(force=True))
    print(build(force=True))
