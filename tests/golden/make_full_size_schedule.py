"""Writes tests/golden/c<k>_full_schedule.txt: the ORACLE's first 100 block steps of config C<k> at its FULL size
(north_star: "active-set and block-time-step indices bit-exact over the first 100 block steps" on all five configs).
The full-size INIT is N^2 pairs -- minutes (C4) to an hour (C5) of host time -- so the result is stored instead of
being recomputed in every test run.  Calls only oracle/ and the seeded input generator.

    python tests/golden/make_full_size_schedule.py 4        # N = 262144, ~5 min on 8 cores
    python tests/golden/make_full_size_schedule.py 5 [threads]   # N = 2^20 + 1, ~1 h on 8 cores

Per block step: t+ (hex float), n_act, CRC-32 of the ascending int32 active list.  After step 100: particle steps,
the per-level histogram, CRC-32 of the t_i and dt_i arrays (float64 bytes), the smallest margin any time-step decision
had to its threshold, and x, v, a, jerk of 64 seeded sample particles (hex floats).
"""
import os
import sys
import zlib

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import oracle  # noqa: E402
from paper_1702_00440_b200 import workloads as W  # noqa: E402

STEPS = 100
SAMPLE_SEED = 4242


def crc(a: np.ndarray) -> int:
    return zlib.crc32(np.ascontiguousarray(a).tobytes()) & 0xFFFFFFFF


def main():
    k = int(sys.argv[1])
    if len(sys.argv) > 2:
        oracle.set_num_threads(int(sys.argv[2]))
    w = W.config(k)
    o = oracle.HermiteOracle(w.m, w.x, w.v, w.eps, w.eta, acc_mode="plain")
    lines = []
    for _ in range(STEPS):
        o.step()
        act = np.asarray(o.active, dtype=np.int32)
        lines.append(f"step {float(o.t).hex()} {len(act)} {crc(act):08x}")
    sample = W.active_indices(w.n, 64, seed=SAMPLE_SEED)
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), f"c{k}_full_schedule.txt")
    with open(out, "w") as f:
        f.write(f"# oracle (oracle/hermite_oracle.c, plain FP64 sums) on workloads.config({k}), N = {w.n}: INIT + the first\n")
        f.write(f"# {STEPS} block steps; written by tests/golden/make_full_size_schedule.py {k}\n")
        f.write("# step <t+ hex> <n_act> <crc32 of the int32 active list>\n")
        f.write("\n".join(lines) + "\n")
        f.write(f"particle_steps {o.particle_steps}\n")
        f.write("level_hist " + " ".join(str(int(c)) for c in o.level_hist) + "\n")
        f.write(f"crc_t {crc(o.t_i):08x}\ncrc_dt {crc(o.dt):08x}\n")
        f.write(f"min_margin {float(o.min_margin)!r}\n")
        f.write(f"nan_count {o.nan_count}\ndtmin_clamps {o.dtmin_clamps}\n")
        f.write(f"# sample <index> then x v a jerk (12 hex floats) after step {STEPS}; indices = active_indices(N, 64, seed={SAMPLE_SEED})\n")
        for i in sample:
            vals = np.concatenate([o.x[i], o.v[i], o.a[i], o.j[i]])
            f.write(f"sample {int(i)} " + " ".join(float(u).hex() for u in vals) + "\n")
    print("wrote", out)


if __name__ == "__main__":
    main()
