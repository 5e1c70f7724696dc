#!/usr/bin/env python
"""bench.py -- the Hermite block-step hot path on synthetic Plummer clusters (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload C2]

One STEP = one pass of the whole hot path over the workload:
    gd_init (a0: all-active force+jerk, initial dt)  ->  gd_energy (a6)
    -> block steps until t_end: gd_next_block (a1), gd_predict (a2), gd_force_jerk (a3/a4),
       gd_correct_and_timestep (a5)  ->  gd_energy (a6)
Default workload: BASELINE.json configs[1] = C2, Plummer sphere N = 16384, eps = 1e-4, eta = 0.01, to t = 1.

metric  = FP64 Hermite force+jerk pair interactions per second (n_act * N per force call, N * N for init);
value   = inputs resident in HBM when the timed region starts;  e2e = same through HOST buffers
          (gd_init_host: H2D of m, x, v inside; gd_get_state_host: D2H of x, v inside).
roofline = the force kernel that took most of the step's time, timed per launch with CUDA events by the library
          ("profile" option) inside the timed region; bound "alu" (plain FP64 FMA pipe, 60 flop per pair).
cpu_baseline / --impl reference = the CPU oracle (oracle/) on the box's host cores, on a bounded sample.

Multi-GPU: the path does not shard in this build (north_star: one GPU) -- "replicas only": every rank runs an
independent replica of the workload; value = sum over ranks / max time over ranks.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time
from pathlib import Path

ROOT = Path(__file__).resolve().parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

FLOP_PER_PAIR = 60.0                      # BASELINE.json convention
ENERGY_FP64_INSTR_PER_PAIR = 13.0         # k_energy_pairs: 3 DADD + 3 DFMA + 5 (rsqrt refinement) + DMUL + DFMA
FP64_NOMINAL_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12   # SMs x DFMA lanes/clk/SM x 2 flop x max SM clock = 37.2
METRIC = "fp64_hermite_force_jerk_interactions_per_s"
UNIT = "interactions/s"


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="C2", help="C1..C5 (BASELINE.json configs); default C2 = configs[1]")
    ap.add_argument("--n", type=int, default=None, help="override the particle count (experiments only)")
    ap.add_argument("--t-end", type=float, default=None, help="override the end time (experiments only)")
    ap.add_argument("--no-sweep", action="store_true", help="skip the C3 force-kernel sweep (extra key)")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--no-c4", action="store_true", help="skip the bounded C4 segment (extra key)")
    ap.add_argument("--no-stages", action="store_true", help="skip the memory-bound stage timing at C5 size (extra key)")
    ap.add_argument("--only-stages", action="store_true", help="run only the memory-bound stage timing (for ncu captures)")
    return ap.parse_args()


def load_workload(args):
    from paper_1702_00440_b200 import workloads as W
    k = int(args.workload.lstrip("Cc"))
    w = W.config(k, n=args.n)
    t_end = args.t_end if args.t_end is not None else w.t_end
    if t_end <= 0.0:
        t_end = 2.0 ** -7                 # C3 names no end time
    return w, t_end


def step_limit(args) -> int:
    """C5 is 'a single all-active force+jerk evaluation plus 10 block steps' (BASELINE.json configs[4])."""
    return 10 if args.workload.lstrip("Cc") == "5" and args.t_end is None else -1


# ------------------------------------------------------------------------------------------- clocks
class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows, self.proc, self.index = [], None, index

    def __enter__(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None
        return self

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def __exit__(self, *exc):
        if self.proc:
            time.sleep(0.25)
            self.proc.terminate()
            self.thread.join(timeout=2)

    def summary(self) -> dict:
        sm, mx, reasons = [], 0.0, set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for r in self.rows:
            try:
                sm.append(float(r[0]))
                mx = max(mx, float(r[1]))
            except (ValueError, IndexError):
                continue
            for name, flag in zip(names, r[3:7]):
                if flag.lower().startswith("active"):
                    reasons.add(name)
        busy = [c for c in sm if c > 0.5 * mx] or sm
        return {"sm_mhz": statistics.median(busy) if busy else None, "sm_max_mhz": mx or None,
                "reasons": sorted(reasons), "samples": len(sm)}


# ------------------------------------------------------------------------------------------ our arm
def run_step(gd, m, x, v, w, t_end, host: bool, profile: bool, max_steps: int = -1, loop_timers: bool = False):
    """One pass of the whole hot path.  host=False: m, x, v are CUDA tensors; host=True: pinned numpy arrays,
    and the final state comes back to host arrays (gd_get_state_host)."""
    h = gd.Hermite(m, x, v, w.eps, w.eta, host=host)
    if profile:
        # gd_init's all-active evaluation runs before the option can be set: the profile pass repeats it once (same
        # kernel, same launch shape, same predicted records at t = 0) so that it is event-timed like the other launches
        import torch
        h.set_option("profile", 1)
        h.predict(0.0)
        h.force_jerk(torch.arange(w.n, dtype=torch.int32, device="cuda"))
    if loop_timers:
        h.set_option("loop_timers", 1)
    k0, u0 = h.energy()
    steps, psteps = h.run_until(t_end, max_steps=max_steps)
    k1, u1 = h.energy()
    out = {"n": w.n, "block_steps": steps, "particle_steps": psteps, "e0": k0 + u0, "e1": k1 + u1,
           "interactions": float(w.n) * w.n + float(psteps) * w.n, "t": h.t}
    if host:
        s = h.state_host(("x", "v"))
        out["d2h_bytes"] = s["x"].nbytes + s["v"].nbytes + 4 * 8       # state + two (K, U) pairs
        out["h2d_bytes"] = 7 * 8 * w.n
    if profile:
        out["prof"] = h.profile()
    out["loop"] = h.loop_profile()
    out["launches"] = h.kernel_launches
    h.close()
    return out


def flush_l2(torch, buf):
    buf.add_(1)                            # 256 MiB read + write: larger than the 126 MB L2


def time_all_active(h, torch, n):
    """One all-active evaluation through gd_force_jerk (all n sinks, explicit list) on the predicted records at t = 0,
    between two CUDA events: the kernel alone, without the host-side setup that gd_init does before it enqueues."""
    idx = torch.arange(n, dtype=torch.int32, device="cuda")
    a = torch.empty((n, 3), dtype=torch.float64, device="cuda")
    j = torch.empty_like(a)
    h.predict(0.0)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record()
    h.force_jerk(idx, a, j)
    e1.record()
    torch.cuda.synchronize()
    return e0.elapsed_time(e1) * 1e-3


def all_active_entry(n, sec, init_s, what):
    return {"n": n, "ms": sec * 1e3, "tflops60": FLOP_PER_PAIR * float(n) * n / sec / 1e12,
            "frac_fp64_nominal": FLOP_PER_PAIR * float(n) * n / sec / 1e12 / FP64_NOMINAL_TFLOPS,
            "gd_init_ms": init_s * 1e3, "what": what}


def warm_allocator(gd, torch, n):
    """The workspace of the next context comes out of torch's caching allocator instead of a cudaMalloc inside a timed
    region (C4: 2 GB): allocate a block of that size once and hand it back to the cache."""
    ws = torch.empty(gd.workspace_bytes(n) + 256, dtype=torch.uint8, device="cuda")
    del ws


def force_sweep(gd, torch, W):
    """C3: isolated gd_force_jerk at N = 65536 over n_act in {1, 16, 256, 4096, 65536} (extra key, not `value`)."""
    w = W.config(3)
    h = gd.Hermite(w.m, w.x, w.v, w.eps, w.eta)
    h.predict(0.0)
    rows = []
    for n_act in (1, 16, 256, 4096, 65536):
        idx = torch.from_numpy(W.active_indices(w.n, n_act)).cuda()
        a = torch.empty((n_act, 3), dtype=torch.float64, device="cuda")
        j = torch.empty_like(a)
        for _ in range(3):
            h.force_jerk(idx, a, j)
        reps = 200 if n_act <= 4096 else 10
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(reps):
            h.force_jerk(idx, a, j)
        e1.record()
        torch.cuda.synchronize()
        sec = e0.elapsed_time(e1) * 1e-3 / reps
        rate = n_act * w.n / sec
        rows.append({"n_act": n_act, "kernel": h.last_force_kernel, "us": round(sec * 1e6, 2),
                     "interactions_per_s": rate, "tflops60": rate * FLOP_PER_PAIR / 1e12,
                     "frac_fp64_nominal": rate * FLOP_PER_PAIR / 1e12 / FP64_NOMINAL_TFLOPS})
    h.close()
    return {"workload": "C3 Plummer N=65536, back-to-back launches (state L2-resident)", "points": rows}


def hbm_peak_gbs() -> tuple[float, str]:
    """Measured copy bandwidth of this pool's B200s (driver-written MEASURED_PEAKS.json), else the recipe's fallback."""
    try:
        return float(json.loads((ROOT / "MEASURED_PEAKS.json").read_text())["hbm_gbs"]), "MEASURED_PEAKS.json hbm_gbs (burst)"
    except (OSError, KeyError, ValueError):
        return 6550.0, "fallback of /opt/skills/guides/B200_PROFILING.md"


def stage_bandwidth(gd, torch, W):
    """The memory-bound stages at C5's size, where the 193 MB state does not fit the
    126 MB L2: next_block (16 B per particle), predictor (184 B per particle: 128 read + 56 written), corrector +
    time step (340 B per active particle).  A shared step (dt_level_min = dt_level_max) makes every block step
    all-active, so the corrector streams all N.  One warm-up step, then one step timed launch by launch with CUDA
    events (extra key, not `value`)."""
    w = W.config(5)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    m_d, x_d, v_d = (torch.from_numpy(u).cuda() for u in (w.m, w.x, w.v))
    warm_allocator(gd, torch, w.n)
    torch.cuda.synchronize()
    e0.record()
    h = gd.Hermite(m_d, x_d, v_d, w.eps, w.eta)      # a0: pack, ONE all-active force+jerk evaluation (N^2 pairs), initial dt
    e1.record()
    torch.cuda.synchronize()
    init_s = e0.elapsed_time(e1) * 1e-3
    eval_s = time_all_active(h, torch, w.n)
    peak, src = hbm_peak_gbs()

    def timed(fn, reps=1):
        torch.cuda.synchronize()
        e0.record()
        for _ in range(reps):
            out = fn()
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) * 1e-3 / reps, out

    rows = {}
    # the usual case first: the first block of C5 under its own block steps (a handful of active particles)
    _, n_first = h.next_block()
    s_nb = statistics.median(timed(h.next_block)[0] for _ in range(9))     # median of nine single calls
    rows["next_block"] = {"us": round(s_nb * 1e6, 2), "n_act": n_first, "algorithmic_bytes": 16.0 * w.n + 4.0 * n_first,
                          "gbs": (16.0 * w.n + 4.0 * n_first) / s_nb / 1e9, "frac_hbm": (16.0 * w.n + 4.0 * n_first) / s_nb / 1e9 / peak,
                          "note": "per call, including the stream synchronisation; the one-kernel form writes (t_next, n_act) into mapped pinned host words itself, so there is no separate device-to-host copy"}
    h.energy()                                         # a6 at this size (warm-up call, then one timed call)
    sec_en, _ = timed(h.energy)
    h.set_option("dt_level_min", 10)
    h.set_option("dt_level_max", 10)
    samples = {"next_block_all_active": [], "predictor": [], "corrector_timestep": []}
    for step in range(4):                              # one warm-up step, three timed: the median is reported
        s_nb, (t_next, n_act) = timed(h.next_block)
        h.predict(t_next)
        s_pr, _ = timed(lambda: h.predict(t_next), 10)
        h.force_jerk(None)
        s_co, _ = timed(h.correct_and_timestep)
        assert n_act == w.n
        if step:
            for name, sec in zip(samples, (s_nb, s_pr, s_co)):
                samples[name].append(sec)
    for name, per in (("next_block_all_active", 20.0), ("predictor", 184.0), ("corrector_timestep", 340.0)):
        sec, nbytes = statistics.median(samples[name]), per * w.n
        rows[name] = {"us": round(sec * 1e6, 2), "algorithmic_bytes": nbytes, "gbs": nbytes / sec / 1e9,
                      "frac_hbm": nbytes / sec / 1e9 / peak}
    h.close()
    rows["next_block_all_active"]["note"] = rows["next_block"]["note"] + "; 4 B of index written per active particle"
    # the predictor's writes (56 B per particle) stay in L2 over back-to-back launches: its DRAM side is the 128 B read
    rows["predictor"]["dram_side_bytes"] = 128.0 * w.n
    rows["predictor"]["frac_hbm_reads_only"] = 128.0 * w.n / (rows["predictor"]["us"] * 1e-6) / 1e9 / peak
    all_active = all_active_entry(w.n, eval_s, init_s, "gd_force_jerk over all N sinks of C5 (N = 2^20 + 1), one call, CUDA events; "
                                  "gd_init_ms = the whole gd_init (host-side setup + pack + the same evaluation + initial dt)")
    # a6 at this size: N (N - 1) / 2 softened pair potentials + N kinetic terms per call (the predictor runs first)
    pairs_en = 0.5 * float(w.n) * (w.n - 1)
    energy = {"n": w.n, "ms": sec_en * 1e3, "pairs_per_s": pairs_en / sec_en,
              "fp64_instr_per_pair": ENERGY_FP64_INSTR_PER_PAIR,
              "frac_fp64_issue": pairs_en * ENERGY_FP64_INSTR_PER_PAIR * 2.0 / sec_en / 1e12 / FP64_NOMINAL_TFLOPS,
              "what": "gd_energy (k_predict + k_energy_pairs + k_energy_reduce + D2H of K, U), one call, CUDA events; fraction = "
                      "pairs x 13 FP64 instructions x 2 flop slots / time / nominal FP64 peak"}
    return {"all_active": all_active, "energy": energy, "workload": f"C5 size N={w.n}, shared step 2^-10 (all-active block steps), median of three steps after a warm-up step; "
                        "predictor: 10 back-to-back launches", "hbm_peak_gbs": peak, "hbm_peak_source": src, "stages": rows}


def c4_segment(gd, torch, W, t_seg=0.125):
    """C4 (BASELINE.json configs[3]: N = 262144, Kroupa-like masses): gd_init event-timed (one all-active evaluation at
    this N), then a bounded segment of its block-step integration -- t = 0 to the first synchronisation time dt_max =
    0.125, half of the config's t = 0.25 -- with the wall time per N-body time unit and the per-level histogram the
    config asks for (extra key, not `value`)."""
    w = W.config(4)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    m_d, x_d, v_d = (torch.from_numpy(u).cuda() for u in (w.m, w.x, w.v))
    warm_allocator(gd, torch, w.n)
    torch.cuda.synchronize()
    e0.record()
    h = gd.Hermite(m_d, x_d, v_d, w.eps, w.eta)
    e1.record()
    torch.cuda.synchronize()
    init_s = e0.elapsed_time(e1) * 1e-3
    eval_s = time_all_active(h, torch, w.n)
    k0, u0 = h.energy()
    h.set_option("loop_timers", 1)          # the per-size bins below need the loop's timers (about 1 % on small steps)
    e0.record()
    steps, psteps = h.run_until(t_seg)
    e1.record()
    torch.cuda.synchronize()
    sec = e0.elapsed_time(e1) * 1e-3
    k1, u1 = h.energy()
    hist, diag = h.level_histogram()
    lp = h.loop_profile()
    sizes = h.loop_histogram()
    h.close()
    pairs = float(psteps) * w.n
    return {
        "all_active": all_active_entry(w.n, eval_s, init_s, "gd_force_jerk over all N sinks of C4 (N = 262144), one call, CUDA events; "
                                       "gd_init_ms = the whole gd_init (host-side setup + pack + the same evaluation + initial dt)"),
        "segment": {"workload": f"C4: {w.name}, eps={w.eps}, eta={w.eta}, block steps t = 0 .. {t_seg} (the first dt_max interval "
                                "of the config's t = 0.25)", "n": w.n, "t_end": t_seg, "ms": sec * 1e3,
                    "wall_s_per_nbody_time_unit": sec / t_seg, "block_steps": steps, "particle_steps": psteps,
                    "interactions_per_s": pairs / sec, "tflops60": FLOP_PER_PAIR * pairs / sec / 1e12,
                    "frac_fp64_nominal": FLOP_PER_PAIR * pairs / sec / 1e12 / FP64_NOMINAL_TFLOPS,
                    "steps_inside_persistent_loop": lp["block_steps"],
                    "energy_rel_err": abs((k1 + u1) / (k0 + u0) - 1.0),
                    "particle_steps_per_level": {str(k): int(c) for k, c in enumerate(hist) if c},
                    "dt_min_clamps": int(diag[1]), "nan_criteria": int(diag[0]),
                    "block_steps_by_active_set_size": [{"n_act_below": r["n_act_below"], "block_steps": r["block_steps"],
                                                        "particle_steps": r["particle_steps"]} for r in sizes]}}


def cpu_sample_steps(n: int) -> int:
    """Block steps in the oracle's bounded sample: about 10-20 s of host work for C2 on 8 cores."""
    return int(min(4096, max(64, (1 << 24) // n)))


def cpu_baseline(w, t_end):
    """The oracle as it stands on the host cores, on a bounded sample of the same workload: INIT (all-active pair
    sums, initial dt) + the first cpu_sample_steps(N) block steps (not past t_end), plain sequential FP64 accumulation."""
    import oracle
    t0 = time.perf_counter()
    o = oracle.HermiteOracle(w.m, w.x, w.v, w.eps, w.eta, acc_mode="plain")
    o.run(t_end, max_steps=cpu_sample_steps(w.n))
    sec = time.perf_counter() - t0
    pairs = float(w.n) * w.n + float(o.particle_steps) * w.n
    return {"value": pairs / sec, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
            "sample": f"{w.name}: INIT (N^2 pairs) + first {o.block_steps} block steps "
                      f"({o.particle_steps} particle steps, to t={o.t:.6g}); plain FP64 sums; {sec:.1f} s"}, sec


def cpu_table(W):
    """the oracle's all-active PAIRSUM rate, single-thread and all cores, at the five sizes (a
    seeded subset of sinks against all N sources where N^2 would take minutes: "subset"), and the share of the
    oracle's block-step run spent in the force sums (the paper: ~95 %).  About 20 s of host work."""
    import numpy as np
    import oracle
    cores = oracle.num_threads()
    rows = []
    for cfg, n_one, n_all in ((1, 1024, 1024), (2, 1024, 8192), (3, 512, 4096), (4, 256, 2048), (5, 128, 1024)):
        w = W.config(cfg)
        row = {"config": f"C{cfg}", "n": w.n}
        for label, k, threads in (("single_thread", n_one, 1), ("all_cores", n_all, cores)):
            k = min(k, w.n)
            idx = None if k == w.n else np.sort(np.random.default_rng(1000 + cfg).choice(w.n, k, replace=False)).astype(np.int32)
            oracle.set_num_threads(threads)
            oracle.pairsum(w.m[:64], w.x[:64], w.v[:64], w.eps, mode="plain")      # the thread team exists before the clock starts
            t0 = time.perf_counter()
            oracle.pairsum(w.m, w.x, w.v, w.eps, idx=idx, mode="plain")
            sec = time.perf_counter() - t0
            row[label] = {"interactions_per_s": k * float(w.n) / sec, "sinks": k, "seconds": round(sec, 3),
                          "sample": "full N^2" if k == w.n else f"subset: {k} seeded sinks x all N sources"}
        oracle.set_num_threads(cores)
        rows.append(row)
    # force share of a block-step run: C1 (N = 1024) to t = 0.125 in full, the oracle's own timers
    w = W.config(1)
    o = oracle.HermiteOracle(w.m, w.x, w.v, w.eps, w.eta, acc_mode="plain")
    o.run(0.125)
    f, tot = o.seconds
    oracle.set_num_threads(1)
    o1 = oracle.HermiteOracle(w.m, w.x, w.v, w.eps, w.eta, acc_mode="plain")
    o1.run(0.125)
    f1, tot1 = o1.seconds
    oracle.set_num_threads(cores)
    return {"cores": cores, "kind": "oracle", "rows": rows,
            "force_share_of_block_step_run": {"workload": "C1 N=1024 to t=0.125 (INIT + %d block steps)" % o.block_steps,
                                              "all_cores": f / tot, "single_thread": f1 / tot1,
                                              "seconds_all_cores": tot, "seconds_single_thread": tot1,
                                              "paper": "~0.95 on a serial CPU build (P:161)"}}


def ncu_traffic(workload: str, kernel: str):
    """dram bytes per launch of `kernel` from the committed `ncu --set full` capture, if profiles/ncu_traffic.csv holds a
    row for this workload and kernel (columns: workload, kernel, dram_bytes, ..., profile, commit; the command that
    made it is in the profile file named there).  A capture is a property of the commit it was taken at, so the row
    names it, together with the kernel's source file and the first 16 hex digits of that file's SHA-256 at the capture:
    `stale` says whether the file in this tree still has that digest (there is no .git on the GPU box to ask).
    No row -> None."""
    try:
        lines = (ROOT / "profiles" / "ncu_traffic.csv").read_text().strip().splitlines()
    except OSError:
        return None, None
    head = lines[0].split(",")
    for ln in lines[1:]:
        row = dict(zip(head, ln.split(",")))
        if row.get("workload") == workload and row.get("kernel") == kernel:
            src = {"profile": row.get("profile"), "commit": row.get("commit"), "stale": None}
            if row.get("source") and row.get("source_sha16"):
                try:
                    import hashlib
                    src["stale"] = hashlib.sha256((ROOT / row["source"]).read_bytes()).hexdigest()[:16] != row["source_sha16"]
                except OSError:
                    pass
            return float(row["dram_bytes"]), src
    return None, None


def aggregate_replicas(torch, dist, device, sec, sec_e2e, pairs, pairs_e2e):
    """Replicas only: the path does not shard, so N ranks run N independent copies of the
    workload with no data-path collective.  The job's time is the MAX over ranks, its work the SUM over ranks.
    dist = None: single process."""
    if dist is None:
        return sec, sec_e2e, pairs, pairs_e2e
    tmax = torch.tensor([sec, sec_e2e], dtype=torch.float64, device=device)
    dist.all_reduce(tmax, op=dist.ReduceOp.MAX)
    work = torch.tensor([pairs, pairs_e2e], dtype=torch.float64, device=device)
    dist.all_reduce(work, op=dist.ReduceOp.SUM)
    return tmax[0].item(), tmax[1].item(), work[0].item(), work[1].item()


def dist_env():
    return int(os.environ.get("RANK", 0)), int(os.environ.get("LOCAL_RANK", 0)), int(os.environ.get("WORLD_SIZE", 1))


def main_ours(args):
    import numpy as np
    import torch
    import torch.distributed as dist
    rank, local_rank, world = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product has no CPU fallback)")
    torch.cuda.set_device(local_rank)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    from paper_1702_00440_b200 import binding as gd, workloads as W
    gd.load()
    if args.only_stages:
        print(json.dumps({"memory_bound_stages": stage_bandwidth(gd, torch, W)}), flush=True)
        return
    w, t_end = load_workload(args)

    # device-resident and pinned-host copies of the inputs
    m_d, x_d, v_d = (torch.from_numpy(u).cuda() for u in (w.m, w.x, w.v))
    m_h, x_h, v_h = (torch.from_numpy(u).pin_memory().numpy() for u in (w.m, w.x, w.v))
    l2buf = torch.zeros(256 << 20, dtype=torch.uint8, device="cuda")

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        run_step(gd, m_d, x_d, v_d, w, t_end, host=False, profile=False, max_steps=step_limit(args))
    run_step(gd, m_h, x_h, v_h, w, t_end, host=True, profile=False, max_steps=step_limit(args))

    # ---- timed region: K steps, inputs resident in HBM, L2 flushed between steps ----
    results = []
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with ClockSampler(local_rank) as clocks:
        barrier()
        e0.record()
        for _ in range(args.steps):
            flush_l2(torch, l2buf)
            results.append(run_step(gd, m_d, x_d, v_d, w, t_end, host=False, profile=False, max_steps=step_limit(args)))
        e1.record()
        barrier()
        # The timed steps replay the captured block-step graph, in which a single launch cannot be bracketed by
        # events.  The per-launch durations come from one more pass of the SAME step, still under the clock sampler,
        # with the library's event timing on: it launches the same kernels directly (the persistent block-step loop,
        # then the stage kernels for any step the loop leaves), each loop / force launch between two events.
        flush_l2(torch, l2buf)
        prof_pass = run_step(gd, m_d, x_d, v_d, w, t_end, host=False, profile=True, max_steps=step_limit(args))
        # and once more with the loop's instantiation that carries device timers (phase split; not the product's kernel)
        prof_pass["loop_timers"] = run_step(gd, m_d, x_d, v_d, w, t_end, host=False, profile=False, max_steps=step_limit(args),
                                            loop_timers=True)["loop"]
    sec = e0.elapsed_time(e1) * 1e-3
    # ---- end to end: K steps through host buffers (H2D of inputs and D2H of the state inside) ----
    e2e_results = []
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        flush_l2(torch, l2buf)
        e2e_results.append(run_step(gd, m_h, x_h, v_h, w, t_end, host=True, profile=False, max_steps=step_limit(args)))
    barrier()
    sec_e2e = time.perf_counter() - t0

    sec, sec_e2e, pairs, pairs_e2e = aggregate_replicas(
        torch, dist if world > 1 else None, "cuda", sec, sec_e2e,
        sum(r["interactions"] for r in results), sum(r["interactions"] for r in e2e_results))
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    return finish_ours(args, gd, W, torch, w, t_end, world, results, e2e_results, sec, sec_e2e, pairs, pairs_e2e,
                       clocks.summary(), prof_pass)


KERNEL_NAMES = {"ipar": "k_force_ipar<2,1>", "jsplit": "k_force_jsplit", "ipar_small": "k_force_ipar<1,4>",
                "loop": "k_block_loop", "slice": "k_force_slice"}


def finish_ours(args, gd, W, torch, w, t_end, world, results, e2e_results, sec, sec_e2e, pairs, pairs_e2e, clocks,
                prof_pass):
    K = args.steps
    prof = {k: {f: prof_pass["prof"][k][f] for f in ("launches", "ms", "pairs")}
            for k in ("ipar", "jsplit", "ipar_small", "loop", "slice")}
    dom = max(prof, key=lambda k: prof[k]["ms"])
    d = prof[dom]
    achieved = FLOP_PER_PAIR * d["pairs"] / (d["ms"] * 1e-3) / 1e12 if d["ms"] > 0 else 0.0
    peak_probe, _ = gd.fp64_peak_probe(1 << 16)
    roofline = {
        "bound": "alu", "kernel": KERNEL_NAMES[dom],
        "achieved": achieved, "peak": FP64_NOMINAL_TFLOPS, "unit": "TFLOP/s", "frac": achieved / FP64_NOMINAL_TFLOPS,
        "traffic": ncu_traffic(args.workload, KERNEL_NAMES[dom])[0],
        "traffic_source": ncu_traffic(args.workload, KERNEL_NAMES[dom])[1],
        "traffic_stale": (ncu_traffic(args.workload, KERNEL_NAMES[dom])[1] or {}).get("stale"),
        "peak_source": "derived: 148 SM x 64 DFMA lanes/clk x 2 flop x 1.965 GHz (MEASURED_PEAKS.json has no FP64 "
                       "entry); register-only DFMA probe on this box: %.2f TFLOP/s" % (peak_probe / 1e12),
        "launches": int(d["launches"]), "avg_launch_us": 1e3 * d["ms"] / max(d["launches"], 1),
        "flop_per_launch": FLOP_PER_PAIR * d["pairs"] / max(d["launches"], 1),
        "share_of_step": d["ms"] * 1e-3 / (sec / K),
        "timing": "per-launch CUDA events (library stream) over one extra pass of the same step with the same kernels "
                  "launched directly; the timed steps replay a captured graph",
        "by_kernel": {k: {"launches": int(v["launches"]), "ms": v["ms"],
                          "tflops60": (FLOP_PER_PAIR * v["pairs"] / (v["ms"] * 1e-3) / 1e12) if v["ms"] > 0 else 0.0}
                      for k, v in prof.items()},
    }
    r0 = results[-1]
    lp = prof_pass["loop_timers"]
    if lp["block_steps"] > 0 and lp["ns"] > 0:
        b = lp["block_steps"]
        # the loop's own device-timer counters (CTA 0's view) over one extra pass with the "loop_timers" option: the
        # timed steps and the event-timed pass run the instantiation without timers
        roofline["loop_timers_pass"] = {
            "block_steps": b, "particle_steps": lp["particle_steps"], "ms": lp["ns"] * 1e-6,
            "tflops60": FLOP_PER_PAIR * lp["particle_steps"] * float(w.n) / (lp["ns"] * 1e-9) / 1e12,
            "us_per_block_step": {"total": lp["ns"] / b * 1e-3, "force": lp["ns_force"] / b * 1e-3,
                                  "wait_partials": lp["ns_barrier1"] / b * 1e-3, "correct": lp["ns_correct"] / b * 1e-3,
                                  "wait_publish": lp["ns_barrier2"] / b * 1e-3}}
    value = pairs / sec
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": args.warmup,
        "ms_per_step": 1e3 * sec / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"{args.workload}: {w.name}, eps={w.eps}, eta={w.eta}, init + block steps "
                               + (f"to t={t_end}" if step_limit(args) < 0 else f"({step_limit(args)} of them)")
                               + " + energy at both ends", "n": w.n, "t_end": t_end,
                   "l2": "256 MiB buffer rewritten between steps (flush); inside a step the %.1f MB state is "
                         "L2-resident by construction" % (184e-6 * w.n),
                   "parallelism": "1 GPU" if world == 1 else f"{world} independent replicas (path does not shard)"},
        "clocks": clocks,
        "e2e": {"value": pairs_e2e / sec_e2e, "unit": UNIT,
                "h2d_bytes_per_step": e2e_results[-1]["h2d_bytes"], "d2h_bytes_per_step": e2e_results[-1]["d2h_bytes"],
                "ms_per_step": 1e3 * sec_e2e / K},
        "gpu_launches": int(sum(r["launches"] for r in results)),
        "roofline": roofline,
        "tflops60": value * FLOP_PER_PAIR / 1e12,
        "frac_fp64_nominal": value * FLOP_PER_PAIR / 1e12 / FP64_NOMINAL_TFLOPS,
        "wall_s_per_nbody_time_unit": (sec / K) / t_end,
        "block_steps": r0["block_steps"], "particle_steps": r0["particle_steps"],
        "mean_n_act": r0["particle_steps"] / max(r0["block_steps"], 1),
        "energy": {"e0": r0["e0"], "e1": r0["e1"], "rel_err": abs(r0["e1"] / r0["e0"] - 1.0)},
    }
    all_active = []
    if not args.no_sweep:
        line["force_sweep"] = force_sweep(gd, torch, W)
        p = line["force_sweep"]["points"][-1]
        all_active.append({"n": 65536, "ms": p["us"] * 1e-3, "tflops60": p["tflops60"], "frac_fp64_nominal": p["frac_fp64_nominal"],
                           "what": "gd_force_jerk over all 65536 sinks of C3, 10 back-to-back launches, CUDA events"})
    if not args.no_c4:
        c4 = c4_segment(gd, torch, W)
        all_active.append(c4["all_active"])
        line["c4_segment"] = c4["segment"]
    if not args.no_stages:
        st = stage_bandwidth(gd, torch, W)
        all_active.append(st.pop("all_active"))
        line["energy_a6"] = st.pop("energy")
        line["memory_bound_stages"] = st
    if all_active:
        # north_star: "the all-active force/jerk kernel sustains >= 70 % of B200 FP64 peak at N >= 65536"
        line["all_active"] = all_active
    if not args.no_cpu and world == 1:
        line["cpu_baseline"], _ = cpu_baseline(w, t_end)
        line["cpu_baseline"]["table"] = cpu_table(W)
    print(json.dumps(line), flush=True)
    return line


# ---------------------------------------------------------------------------------------- reference arm
def main_reference(args):
    """The oracle as it stands, timed on the host cores: each step = the bounded sample of cpu_baseline()."""
    rank, _, world = dist_env()
    if rank != 0:
        return
    w, t_end = load_workload(args)
    for _ in range(min(args.warmup, 1)):              # a CPU program needs no more than one warm-up pass
        cpu_baseline(w, t_end)
    secs, vals, info = 0.0, [], None
    for _ in range(args.steps):
        info, s = cpu_baseline(w, t_end)
        secs += s
        vals.append(info["value"])
    value = sum(vals) / len(vals)
    info = dict(info, value=value)
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * secs / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"{args.workload}: {w.name}, eps={w.eps}, eta={w.eta}; bounded sample per step: "
                                   f"INIT + first {cpu_sample_steps(w.n)} block steps", "n": w.n, "t_end": t_end},
            "cpu_baseline": info,
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


if __name__ == "__main__":
    a = parse_args()
    if a.impl == "reference":
        main_reference(a)
    else:
        main_ours(a)
