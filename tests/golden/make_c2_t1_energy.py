"""Writes tests/golden/c2_t1_energy.txt: the ORACLE's result for config C2 (Plummer N = 16384, eps = 1e-4, eta = 0.01)
integrated to t = 1 -- block steps, particle steps, E(0), E(1).  Calls only oracle/ and the seeded input generator;
about 5 minutes on 8 cores (1.13e11 pair interactions, plain FP64 sums).

    python tests/golden/make_c2_t1_energy.py
"""
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import oracle  # noqa: E402
from paper_1702_00440_b200 import workloads as W  # noqa: E402

w = W.config(2)
o = oracle.HermiteOracle(w.m, w.x, w.v, w.eps, w.eta, acc_mode="plain")
k0, u0 = o.energy()
o.run(1.0)
k1, u1 = o.energy()
with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "c2_t1_energy.txt"), "w") as f:
    f.write("# oracle (oracle/hermite_oracle.c, plain FP64 sums) on workloads.config(2) to t = 1; north_star: the same\n")
    f.write("# |dE/E| to within 10 % after one N-body time unit; written by tests/golden/make_c2_t1_energy.py\n")
    f.write(f"block_steps {o.block_steps}\nparticle_steps {o.particle_steps}\n")
    f.write(f"e0 {k0 + u0!r}\ne1 {k1 + u1!r}\n")
