"""Test and bench harness (not part of the shipped library): seeded synthetic workloads of BASELINE.json:configs
(workloads.py — generators, ghost fill, group cutting, the R15 time step; none of the method's arithmetic), the R14
error metric (metrics.py) and the GPU-vs-oracle comparison with the R7 guard accounting (parity.py)."""
