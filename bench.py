#!/usr/bin/env python
"""bench.py -- throughput of the MPC hot path (BASELINE.json metric: particle-updates/s on one B200
and achieved HBM GB/s vs the roofline).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg5] [--nbar 10] [--impl reference]

A "step" is one full MPC step (stream, shift, key, [reorder], cell sums, cell finalize, collide) over
all particles of the workload. Default workload = BASELINE.json configs[4] ("cfg5"): SRD, 512^3
cells, 10 particles/cell (1.342e9 particles, 32 GB of fp32 state), alpha = 130 deg, dt = 0.1,
k_BT = 1 cell thermostat, reorder every 10 steps. Inputs are seeded synthetic (uniform positions,
Maxwell velocities; paper_2406_15236_b200/inputs.py) and far larger than L2, so nothing is flushed
between steps. N > 1 (under torchrun) runs N independent replicas, one per GPU ("replicas only",
DESIGN.md): no data-path collective, `value` = all ranks' particle-updates / max-over-ranks time.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

WORKLOADS = {
    # name: (cells, nbar, params, default steps, default warmup)
    "cfg1": dict(cells=(16, 16, 16), nbar=10, kw=dict(), rebin_every=1),
    "cfg2": dict(cells=(64, 64, 64), nbar=10, kw=dict(thermostat=1), rebin_every=1),
    "cfg3": dict(cells=(128, 128, 128), nbar=10, kw=dict(collision=1, conserve_L=1, dt=0.02), rebin_every=1),
    # config 4 does not name a reorder interval: 10, the value of its full-length test (tests/test_configs_freerun_gpu.py)
    "cfg4": dict(cells=(256, 64, 64), nbar=10, kw=dict(thermostat=1, bc=(0, 0, 1), g=(0.001, 0, 0)), rebin_every=10),
    "cfg5": dict(cells=(512, 512, 512), nbar=10, kw=dict(thermostat=1), rebin_every=10),
}
# algorithmic bytes per particle-step (SURVEY.md 8d / DESIGN.md "Roofline"): read r,v 24 B + write r,v 24 B
# + per-cell record written once and read once (SRD+MBS: 20 B each way) -> 48 + 40/<N_c>
def algorithmic_bytes_per_update(nbar, collision=0, conserve_L=0):
    if collision == 1 or conserve_L:
        return 48.0 + (88.0 + 48.0) / nbar
    return 48.0 + 40.0 / nbar


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """SM clock and throttle reasons during the timed region: ONE `nvidia-smi -lms 50` process streams a line every 50 ms
    (starting a new nvidia-smi per sample takes longer than the whole timed region of a short run); it is started before the
    warm-up, and mark_start() / mark_stop() around the timed region pick the lines that fall inside it. `samples` is that
    number: below 5 the record cannot support a statement about the clock, and says so."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")
    PERIOD_MS = 50

    def __init__(self, index):
        self.index, self.rows, self._t, self._p = index, [], None, None
        self.t0 = self.t1 = None

    def _run(self):
        try:
            for line in self._p.stdout:
                cols = [t.strip() for t in line.strip().split(",")]
                if len(cols) >= 7:
                    self.rows.append((time.monotonic(), cols))
        except Exception:
            pass

    def __enter__(self):
        try:
            self._p = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                        "-lms", str(self.PERIOD_MS)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True, bufsize=1)
            self._t = threading.Thread(target=self._run, daemon=True)
            self._t.start()
        except Exception:
            self._p = None
        return self

    def mark_start(self):
        self.t0 = time.monotonic()

    def mark_stop(self):
        self.t1 = time.monotonic()

    def __exit__(self, *a):
        if self._p is not None:
            self._p.terminate()
            try:
                self._p.wait(timeout=5)
            except Exception:
                self._p.kill()
            self._t.join(timeout=5)

    def summary(self):
        num = lambda t: t.replace(".", "", 1).isdigit()
        inside = [c for (t, c) in self.rows if self.t0 is not None and self.t1 is not None and self.t0 <= t <= self.t1]
        sm = [float(c[0]) for c in inside if num(c[0])]
        mx = [float(c[1]) for (_, c) in self.rows if num(c[1])]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = sorted({names[i] for c in inside for i in range(4) if c[3 + i].lower().startswith("active")})
        out = {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None, "reasons": reasons,
               "samples": len(inside), "sample_period_ms": self.PERIOD_MS, "samples_outside_timed_region": len(self.rows) - len(inside)}
        if len(inside) < 5:
            out["note"] = "fewer than 5 samples inside the timed region: insufficient for a statement about the clock under load"
        return out


def oracle_rate(wl, nbar, budget_s=12.0):
    """The CPU oracle, as it stands, on a bounded sample of the workload: same parameters on a 64^3-cell
    box (or the workload itself if smaller), single thread. Returns (updates/s, description, steps)."""
    from oracle.binding import Oracle
    from paper_2406_15236_b200.inputs import uniform_maxwell

    cells = tuple(min(c, 64) for c in wl["cells"])
    box = tuple(float(c) for c in cells)
    n = int(np.prod(cells)) * nbar
    kw = dict(wl["kw"])
    kw.update(rebin_every=wl["rebin_every"], brick=1)
    o = Oracle(box, cells, nbar, 1234, **kw)
    o.set_state(*uniform_maxwell(box, n, 1234))
    t0 = time.perf_counter()
    o.step(1)
    t1 = time.perf_counter() - t0
    steps = int(max(2, min(200, budget_s / max(t1, 1e-6))))
    t0 = time.perf_counter()
    o.step(steps)
    dt = time.perf_counter() - t0
    return n * steps / dt, f"{cells[0]}x{cells[1]}x{cells[2]} cells x {nbar}/cell ({n} particles), {steps} steps, same parameters", steps, dt / steps


def max_over_ranks(dist, ms, device):
    """Replicas only: the only exchange between ranks is this MAX of the device-timed
    milliseconds (and the barriers around the timed region)."""
    if dist is None:
        return float(ms)
    import torch

    t = torch.tensor([ms], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_rate(world, n_per_rank, steps, ms):
    """Whole-job particle-updates/s: every rank advances its own replica of n_per_rank particles (weak scaling)."""
    return world * n_per_rank * steps / (ms * 1e-3)


def run_reference(args, wl, rank, world):
    if rank != 0:
        return
    nbar = args.nbar
    cells = tuple(min(c, 64) for c in wl["cells"])
    from oracle.binding import Oracle
    from paper_2406_15236_b200.inputs import uniform_maxwell
    box = tuple(float(c) for c in cells)
    n = int(np.prod(cells)) * nbar
    kw = dict(wl["kw"])
    kw.update(rebin_every=wl["rebin_every"], brick=1)
    o = Oracle(box, cells, nbar, 1234, **kw)
    o.set_state(*uniform_maxwell(box, n, 1234))
    o.step(args.warmup)
    t0 = time.perf_counter()
    o.step(args.steps)
    dt = time.perf_counter() - t0
    val = n * args.steps / dt
    sample = f"{cells[0]}x{cells[1]}x{cells[2]} cells x {nbar}/cell ({n} particles) per step, same parameters as the workload"
    line = {"impl": "reference", "metric": "MPC particle-updates/sec", "value": val, "unit": "particle-updates/s",
            "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": args.workload, "cells": list(wl["cells"]), "n_per_cell": nbar,
                       "note": "CPU oracle (oracle/mpc_oracle.cpp, single thread) timed on a bounded sample of the workload"},
            "cpu_baseline": {"value": val, "unit": "particle-updates/s", "cores": 1, "host_cores": os.cpu_count(), "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": "particle-updates/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def csrc_digest():
    """sha256 over every CUDA source of the library (all of them decide what a step launches): ties a committed ncu
    capture to the code it was taken from."""
    import hashlib
    h = hashlib.sha256()
    d = os.path.join(ROOT, "paper_2406_15236_b200", "csrc")
    for f in sorted(os.listdir(d)):
        if f.endswith((".cu", ".cuh")):
            h.update(f.encode())
            h.update(open(os.path.join(d, f), "rb").read())
    return h.hexdigest()[:16]


def captured_traffic(family, workload, nbar):
    """DRAM bytes per launch (dram__bytes_read.sum + dram__bytes_write.sum) of a kernel family from the committed
    `ncu --set full` capture (profiles/traffic.json, written by hand from the capture named there). Returns
    (bytes or None, source, stale): stale = the capture was taken from other CUDA sources than the ones built now."""
    p = os.path.join(ROOT, "profiles", "traffic.json")
    if not os.path.exists(p):
        return None, None, None
    t = json.load(open(p))
    e = t.get("kernels", {}).get(f"{family}:{workload}:nbar{nbar}")
    if e is None:
        return None, None, None
    return float(e["dram_bytes_per_launch"]), e.get("source"), e.get("csrc_digest") != csrc_digest()


def measure(args, workload, nbar, steps, warmup, rank, local_rank, world, dist, with_e2e, rebin_every=None):
    """One workload: W untimed warm-up steps, then EXACTLY K steps in one mpc_step call between two CUDA events on
    the launching stream. Returns the JSON-able result dict (without cpu_baseline)."""
    import torch

    from paper_2406_15236_b200 import MPC
    from paper_2406_15236_b200.inputs import uniform_maxwell_cuda

    wl = dict(WORKLOADS[workload])
    if rebin_every is not None:
        wl["rebin_every"] = rebin_every
    device = torch.device(f"cuda:{local_rank}")
    cells = wl["cells"]
    box = tuple(float(c) for c in cells)
    n = int(np.prod(cells)) * nbar
    kw = dict(wl["kw"])
    brick = tuple(int(t) for t in args.brick.split(","))
    brick = brick * 3 if len(brick) == 1 else brick
    kw.update(rebin_every=wl["rebin_every"], brick=brick)
    compact = n * 72 + int(np.prod(cells)) * 80 > 150e9
    # a state that does not fit beside the workspace (20 per cell: 64 GB + 138 GB) is made array by array on the
    # device, parked in pinned host memory and handed over through the host-pointer ABI
    via_host = n * 24 + n * 52 + int(np.prod(cells)) * 80 > 170e9
    st = list(uniform_maxwell_cuda(box, n, 1234 + rank, device=str(device), to_host=via_host))
    torch.cuda.empty_cache()
    sim = MPC(box, cells, nbar, 1234 + rank, n_max=n, device=str(device), compact=compact, **kw)
    if via_host:
        sim.set_state_host(*st)
    else:
        sim.set_state(*st)
    torch.cuda.synchronize()
    del st
    sim._keep = None
    torch.cuda.empty_cache()

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
            torch.cuda.synchronize()

    # ---- warm-up (untimed), then EXACTLY K timed steps, CUDA events on the launching stream ----
    # The collision of the last step of a call stays pending and is applied inside the next call's first streaming
    # pass: the timed call applies the warm-up's last collision and leaves its own last one pending,
    # i.e. exactly K collisions, K streaming passes, K cell passes are inside the timed region.
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with ClockSampler(local_rank) as clocks:     # streaming from before the warm-up on
        sim.step(warmup)
        barrier()
        sim.profile_enable(True)
        sim.profile_read()
        l0 = sim.launch_count
        barrier()
        clocks.mark_start()
        ev0.record(sim.stream)
        sim.step(steps)
        ev1.record(sim.stream)
        barrier()
        clocks.mark_stop()
    ms = ev0.elapsed_time(ev1)
    launches = sim.launch_count - l0
    prof = sim.profile_read()
    sim.profile_enable(False)
    ms = max_over_ranks(dist, ms, device)
    ob = sim.observables()
    value = whole_job_rate(world, n, steps, ms)

    # ---- roofline of the dominant kernel family (live CUDA-event times from the timed region) ----
    peak, peak_src = measured_peaks()
    balg = algorithmic_bytes_per_update(nbar, kw.get("collision", 0), kw.get("conserve_L", 0))
    fam = {k: v for k, v in prof.items() if v[1] > 0}
    total_fam_ms = sum(v[0] for v in fam.values())
    dom = max(fam, key=lambda k: fam[k][0]) if fam else None
    roofline = None
    if dom:
        dms, dcnt = fam[dom]
        fam_bytes = kernel_algorithmic_bytes(dom, n, int(np.prod(cells)), nbar)
        ach = fam_bytes / (dms / dcnt * 1e-3) / 1e9
        traffic, tsrc, stale = captured_traffic(dom, workload, nbar)
        roofline = {"bound": "hbm", "kernel": dom, "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak,
                    "traffic": traffic, "traffic_source": tsrc, "traffic_capture_is_of_other_sources": stale,
                    "peak_source": peak_src, "avg_ms": dms / dcnt, "launches_timed": dcnt,
                    "algorithmic_bytes_per_launch": fam_bytes,
                    "step_frac_of_roofline": value / world * balg / 1e9 / peak,
                    "step_frac_of_8000": value / world * balg / 1e9 / 8000.0,
                    "family_ms_per_step": {k: v[0] / steps for k, v in sorted(fam.items(), key=lambda kv: -kv[1][0])},
                    "family_share": {k: v[0] / total_fam_ms for k, v in fam.items()}}
    res = {"value": value, "ms_per_step": ms / steps, "steps": steps, "warmup": warmup, "gpu_launches": int(launches),
           "clocks": clocks.summary(), "roofline": roofline,
           "config": {"workload": workload, "cells": list(cells), "n_per_cell": nbar, "particles": n,
                      "collision": "MPC-AT" if kw.get("collision") else "SRD", "conserve_L": bool(kw.get("conserve_L", 0)),
                      "thermostat": bool(kw.get("thermostat", 0)),
                      "rebin_every": wl["rebin_every"], "brick": list(brick), "compact_workspace": bool(compact),
                      "l2": "inputs larger than L2 (no flush)" if n * 24 > 4 * 126e6 else ("state fits in L2 (L2-resident, launch-bound): HBM fraction not meaningful" if n * 24 < 126e6 else "state within 4x L2 (partly L2-resident): HBM fraction not meaningful"),
                      "parallelism": "replicas only" if world > 1 else "single GPU",
                      "algorithmic_bytes_per_update": balg,
                      "collisions_in_timed_region": "K (the warm-up's last collision is applied by the first timed sweep, the last timed one stays pending)"},
           "check": {"kT_cell": ob["kT_cell"], "kT_est": ob["kT_est"], "max_cell_count": ob["max_cell_count"], "step": ob["step"],
                     "n_range_overflows": ob["n_range_overflows"]}}
    if with_e2e:
        res["e2e"] = run_e2e(sim, n, steps)
    sim.close()
    del sim
    torch.cuda.empty_cache()
    return res, wl


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=30)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--workload", default="cfg5", choices=sorted(WORKLOADS))
    ap.add_argument("--nbar", type=int, default=None, help="particles per cell (cfg5 sweep: 5, 10, 20)")
    ap.add_argument("--brick", default="16,16,8", help="brick dims of the memory key, e.g. 16,16,8")
    ap.add_argument("--rebin-every", type=int, default=None)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-extras", action="store_true", help="skip the density sweep and the other workloads")
    args = ap.parse_args()
    wl = dict(WORKLOADS[args.workload])
    explicit = args.nbar is not None or args.workload != "cfg5" or args.rebin_every is not None
    if args.nbar is None:
        args.nbar = wl["nbar"]
    if args.rebin_every is not None:
        wl["rebin_every"] = args.rebin_every
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))

    if args.impl == "reference":
        run_reference(args, wl, rank, world)
        return

    import torch

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product has no CPU fallback")
    dist = None
    if world > 1:
        import torch.distributed as dist
        torch.cuda.set_device(local_rank)
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local_rank}"))
    torch.cuda.set_device(torch.device(f"cuda:{local_rank}"))

    res, wl = measure(args, args.workload, args.nbar, args.steps, args.warmup, rank, local_rank, world, dist,
                      with_e2e=(not args.no_e2e and rank == 0 and world == 1), rebin_every=args.rebin_every)
    line = {"metric": "MPC particle-updates/sec", "value": res["value"], "unit": "particle-updates/s", "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": res["ms_per_step"], "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": res["config"], "gpu_launches": res["gpu_launches"], "clocks": res["clocks"], "roofline": res["roofline"],
            "check": res["check"]}
    line["e2e"] = res.get("e2e") if world == 1 else None

    # ---- extras of the default run (N = 1): the density sweep BASELINE.json configs[4] names, and configs 3 and 4 ----
    if world == 1 and rank == 0 and not explicit and not args.no_extras:
        sweep = []
        for nb in (5, 20):
            r, _ = measure(args, "cfg5", nb, args.steps, args.warmup, rank, local_rank, world, None, with_e2e=False)
            sweep.append({"n_per_cell": nb, "particles": r["config"]["particles"], "ms_per_step": r["ms_per_step"], "value": r["value"],
                          "step_frac_of_roofline": r["roofline"]["step_frac_of_roofline"], "step_frac_of_8000": r["roofline"]["step_frac_of_8000"],
                          "compact_workspace": r["config"]["compact_workspace"], "clocks": r["clocks"],
                          "family_ms_per_step": r["roofline"]["family_ms_per_step"], "check": r["check"]})
        line["density_sweep"] = sweep
        other = []
        # configs 1 and 2 (40,960 and 2.6e6 particles) live in L2 and are bound by kernel launches, not by HBM: reported
        # as updates/s, their "fraction of the HBM roofline" means nothing and is flagged in config.l2
        for w, k in (("cfg1", 1000), ("cfg2", 300), ("cfg3", 100), ("cfg4", 100)):
            r, _ = measure(args, w, WORKLOADS[w]["nbar"], k, 10, rank, local_rank, world, None, with_e2e=False)
            other.append({"workload": w, "config": r["config"], "ms_per_step": r["ms_per_step"], "value": r["value"],
                          "steps": k, "gpu_launches": r["gpu_launches"],
                          "step_frac_of_roofline": r["roofline"]["step_frac_of_roofline"],
                          "family_ms_per_step": r["roofline"]["family_ms_per_step"], "check": r["check"]})
        line["other_workloads"] = other
    # ---- CPU oracle beside it (rank 0, N = 1 only) ----
    if not args.no_cpu_baseline and rank == 0 and world == 1:
        v, sample, _, _ = oracle_rate(wl, args.nbar)
        line["cpu_baseline"] = {"value": v, "unit": "particle-updates/s", "cores": 1, "host_cores": os.cpu_count(),
                                "kind": "oracle", "sample": sample}
    if rank == 0:
        print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


def kernel_algorithmic_bytes(family, n, ncells, nbar):
    """Algorithmic bytes one launch of a kernel family must move."""
    per_particle = {"stream_key": 24 + 12 + 4, "accum": 12 + 4, "collide": 12 + 4 + 12, "gather": 4 + 32 + 32,
                    "scatter_slots": 8 + 8, "rank": 12 + 4, "sweep": 48, "sweep_gather": 48 + 32 / 3.0}.get(family, 0)
    # sweep: the per-cell record is read once (32 B) and the cell sums written once (20 B of payload)
    per_cell = {"accum": 20, "cell": 20 + 32, "collide": 32, "scan": 8, "memset": 24, "sweep": 20 + 20, "sweep_gather": 20 + 20}.get(family, 0)
    return float(per_particle) * n + float(per_cell) * ncells


def run_e2e(sim, n, steps):
    import torch

    host = [torch.empty(n, dtype=torch.float32, pin_memory=True) for _ in range(6)]
    hid = torch.empty(n, dtype=torch.int32, pin_memory=True)
    sim.get_state_host(out=host + [hid])                   # current state -> pinned host buffers (untimed)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    sim.set_state_host(*host, id=hid, step=0)              # H2D inside the timed region
    sim.step(steps)
    ob = sim.observables()                                 # D2H of the step result (synchronises)
    sim.get_state_host(out=host + [hid])                   # D2H of the final state
    dt = time.perf_counter() - t0
    del ob
    return {"value": n * steps / dt, "unit": "particle-updates/s", "h2d_bytes_per_step": 28.0 * n / steps,
            "d2h_bytes_per_step": 28.0 * n / steps, "seconds": dt, "steps": steps,
            "note": "one job = mpc_set_state_host (pinned) + mpc_step(K) + mpc_observables + mpc_get_state_host"}


if __name__ == "__main__":
    main()
