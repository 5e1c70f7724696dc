"""Writes tests/golden/c2_t1_energy.txt (default) or c2_t1_energy_single_halving.txt (--halving-mode 0): the ORACLE's
result for config C2 (Plummer N = 16384, eps = 1e-4, eta = 0.01) integrated to t = 1 -- block steps, particle steps,
E(0), E(1) -- under one of the two readings of the block rule (R7):
    halving mode 1 (the default of the oracle and of the CUDA path): dt_req < h -> halve until dt <= dt_req;
    halving mode 0: a single halving per step.
The pair of files is what tests/test_oracle_integrator.py::test_block_rule_reading_against_the_papers_energy_error
reads: only the first reading reaches the accuracy the paper states for eta = 0.01 (dE/E0 ~ 1e-7).
Calls only oracle/ and the seeded input generator; about 5 minutes per mode on 8 cores (1.13e11 pair interactions,
plain FP64 sums).

    python tests/golden/make_c2_t1_energy.py [--halving-mode 0|1]
"""
import argparse
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import oracle  # noqa: E402
from paper_1702_00440_b200 import workloads as W  # noqa: E402

ap = argparse.ArgumentParser()
ap.add_argument("--halving-mode", type=int, default=1, choices=[0, 1])
mode = ap.parse_args().halving_mode

w = W.config(2)
o = oracle.HermiteOracle(w.m, w.x, w.v, w.eps, w.eta, halving_mode=mode, acc_mode="plain")
k0, u0 = o.energy()
o.run(1.0)
k1, u1 = o.energy()
name = "c2_t1_energy.txt" if mode == 1 else "c2_t1_energy_single_halving.txt"
with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), name), "w") as f:
    f.write("# oracle (oracle/hermite_oracle.c, plain FP64 sums) on workloads.config(2) to t = 1; north_star: the same\n")
    f.write("# |dE/E| to within 10 % after one N-body time unit; written by tests/golden/make_c2_t1_energy.py\n")
    if mode == 0:
        f.write("# halving mode 0 (a single halving per step): the reading of the block rule that DESIGN.md R7 does NOT take\n")
    f.write(f"block_steps {o.block_steps}\nparticle_steps {o.particle_steps}\n")
    f.write(f"e0 {k0 + u0!r}\ne1 {k1 + u1!r}\n")
print(name, o.block_steps, o.particle_steps, abs((k1 + u1) / (k0 + u0) - 1.0))
