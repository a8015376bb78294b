#!/usr/bin/env python
"""bench.py - throughput of the cable-step hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--mode stream|fused]

Workload: BASELINE.json configs[3] ("C3 large": 100,000 cells, depth-6 trees of 63 branches x 8
control volumes, ~5.05e7 CVs, 50 exponential synapses and 50 incoming connections per cell,
dt = 0.025 ms), seeded and synthetic (paper_1901_07454_b200.workloads.config3, driven variant).

A bench "step" is ONE MINIMUM-DELAY EPOCH of that network: 200 grid steps of dt (5 ms of simulated
time; event delivery, mechanism currents, matrix assembly, Hines solve, voltage update, state update
and threshold test 200 times - rows a0..a6 of SURVEY.md 8(a)) followed by the epoch boundary that
turns the epoch's spikes into queued events (row a7).  metric = compartment-steps/s =
(number of CVs) x (grid steps) / device time of arb_advance.

mode "stream" (default, the headline): one cable-step kernel launch per grid step, every cell's
state and coefficients stream through HBM each step - the configuration SURVEY.md 8(d) defines the
level-A HBM roofline for.  mode "fused": the same kernel keeps a cell's state on chip for a whole
epoch (ARB_OPT_FUSED_STEPS = 0); reported beside the headline under "fused_epoch".

N > 1 (torchrun): the path shards by cells with no data-path collective:
every rank integrates its own closed 100,000-cell network (cells first_cell = rank * 100000 ...
of the same population), weak scaling; value = CV-steps of all ranks / max-over-ranks device time.

--impl reference: times the CPU oracle (oracle/, plain fp64 C, as it stands) on this box's host
cores on a bounded sample of the same workload; rank 0 only.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "compartment-steps/sec (fp64), C3 100k cells"
UNIT = "CV-steps/s"
EPOCH_MS = 5.0          # minimum connection delay of configs[3] is U(5,10) ms -> epochs of 200 steps
DT = 0.025
STEPS_PER_EPOCH = 200
FALLBACK_HBM_GBS = 6650.0   # /opt/skills/guides/B200_PROFILING.md fallback


# --------------------------------------------------------------------------------------------
# helpers
# --------------------------------------------------------------------------------------------
def measured_peak_hbm():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


def algorithmic_bytes_per_grid_step(m):
    """Level-A bytes one grid step must move:
    48 B per CV (V read + write, rhs coefficients a,b, solver factors f, 1/d), 4 B per branch
    (parent link), 80 B per HH CV (m,h,n read + write, three conductances, slot), 20 B per synapse
    (g read + write, CV index)."""
    off = m["cv_off"]
    par = m["cv_parent"].astype(np.int64)
    base = np.repeat(off[:-1], np.diff(off))
    gpar = np.where(par >= 0, par + base, -1)
    nchild = np.bincount(gpar[gpar >= 0], minlength=m["n_cv"])
    starts = (gpar < 0) | (nchild[np.maximum(gpar, 0)] != 1)
    n_branch = int(np.count_nonzero(starts))
    n_hh = 0
    if m["hh_gnabar"] is not None:
        n_hh = int(np.count_nonzero((m["hh_gnabar"] != 0) | (m["hh_gkbar"] != 0) | (m["hh_gl"] != 0)))
    return 48 * m["n_cv"] + 4 * n_branch + 80 * n_hh + 20 * m["n_syn"]


def committed_traffic(kernel):
    """dram bytes per launch of `kernel` from the committed ncu capture (profiles/roofline_traffic.csv)."""
    p = os.path.join(ROOT, "profiles", "roofline_traffic.csv")
    try:
        with open(p) as f:
            for line in f:
                c = [x.strip() for x in line.split(",")]
                if len(c) >= 3 and c[0] == kernel:
                    return float(c[2])
    except Exception:
        pass
    return None


class ClockSampler:
    """nvidia-smi clocks / throttle reasons while the timed region runs (B200_PROFILING.md)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index):
        self.idx, self.proc, self.lines = gpu_index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.idx), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line)

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for line in self.lines:
            c = [x.strip() for x in line.split(",")]
            if len(c) < 9:
                continue
            try:
                sm.append(float(c[1])), mx.append(float(c[2])), pw.append(float(c[3]))
            except ValueError:
                continue
            for nm, v in zip(names, c[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(mx)), "power_w_max": float(max(pw)),
                "samples": len(sm), "reasons": sorted(reasons)}


def dist_env():
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    return rank, world, local


def reduce_over_ranks(elapsed_ms, units, world, backend_device):
    """Whole-job figures from per-rank ones: MAX of the device times, SUM of the units processed.
    Uses torch.distributed when world > 1 (nccl on the GPU box, gloo in the CPU test)."""
    if world == 1:
        return float(elapsed_ms), float(units)
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(elapsed_ms)], dtype=torch.float64, device=backend_device)
    u = torch.tensor([float(units)], dtype=torch.float64, device=backend_device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


# --------------------------------------------------------------------------------------------
# reference arm / cpu_baseline: the oracle on the host cores
# --------------------------------------------------------------------------------------------
def oracle_sample(n_cells_sample, first_cell=0):
    """First `n_cells_sample` cells of the C3 population as an isolated network (their external
    events kept, connections dropped): the same per-cell work as in the full network."""
    from paper_1901_07454_b200 import workloads as W
    m = W.config3(n_cells=n_cells_sample + 1, first_cell=first_cell)
    return W.take_cells(m, np.arange(n_cells_sample))


def time_oracle(sample_cells, steps, warmup, threads=None):
    from oracle import orc
    orc.build()
    cores = threads or os.cpu_count() or 1
    sub = oracle_sample(sample_cells)
    o = orc.Oracle(sub, threads=cores)
    t = 0.0
    times = []
    for i in range(warmup + steps):
        t0 = time.perf_counter()
        t += EPOCH_MS
        o.advance(t, DT)
        dt_ = time.perf_counter() - t0
        if i >= warmup:
            times.append(dt_)
    o.close()
    per_step = float(np.mean(times))
    return dict(value=sub["n_cv"] * STEPS_PER_EPOCH / per_step, ms_per_step=per_step * 1e3, cores=cores,
                sample="first %d cells of C3 (%d CVs, connections dropped, external events kept), "
                       "%d epochs of 200 steps, %s" % (sample_cells, sub["n_cv"], steps,
                                                       "OpenMP over cells" if cores > 1 else "one thread"))


def run_reference(args):
    rank, world, _ = dist_env()
    if rank != 0:
        return
    r = time_oracle(args.ref_cells, args.steps, min(args.warmup, 1))
    line = {"impl": "reference", "metric": METRIC, "value": r["value"], "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": min(args.warmup, 1), "ms_per_step": r["ms_per_step"],
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic",
            "config": {"workload": "configs[3] C3 large (bounded sample: %s)" % r["sample"]},
            "cpu_baseline": {"value": r["value"], "unit": UNIT, "cores": r["cores"], "kind": "oracle",
                             "sample": r["sample"]},
            "e2e": {"value": r["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# --------------------------------------------------------------------------------------------
# our arm
# --------------------------------------------------------------------------------------------
def timed_epochs(torch, g, t_now, n, sync_all):
    """n epochs through arb_advance, device time by CUDA events on the model's stream."""
    sync_all()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(g.stream)
    for _ in range(n):
        t_now += EPOCH_MS
        g.advance(t_now, DT)
    e1.record(g.stream)
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1)
    sync_all()
    return ms, t_now


def run_ours(args):
    import torch
    rank, world, local = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the hot path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    def sync_all():
        if world > 1:
            torch.distributed.barrier()
        torch.cuda.synchronize()

    from paper_1901_07454_b200 import binding as B, workloads as W
    B.lib()
    m = W.config3(n_cells=args.cells, first_cell=rank * args.cells)
    g = B.Model(m, device="cuda:%d" % local)
    fused_steps = {"stream": 1, "fused": 0}
    g.set_option(B.ARB_OPT_FUSED_STEPS, fused_steps[args.mode])
    n_cv = m["n_cv"]
    units_per_step = n_cv * STEPS_PER_EPOCH

    # ---- device-resident timing: W warm-up epochs, K timed epochs
    t_now = 0.0
    _, t_now = timed_epochs(torch, g, t_now, args.warmup, sync_all)
    g.set_option(B.ARB_OPT_TIMING, 1)
    st0 = g.stats()
    l0 = st0["launches"]
    sub0 = g.probe(B.ARB_PROBE_NSTEPS)
    spikes0 = int(B.lib().arb_spikes(g._h, None, None, 0))
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    ms, t_now = timed_epochs(torch, g, t_now, args.steps, sync_all)
    clocks = sampler.stop() if rank == 0 else None
    tim = g.timing()
    g.set_option(B.ARB_OPT_TIMING, 0)
    st1 = g.stats()
    launches = st1["launches"] - l0
    n_events = st1["events_delivered"] - st0["events_delivered"]
    sub1 = g.probe(B.ARB_PROBE_NSTEPS)
    n_spikes = int(B.lib().arb_spikes(g._h, None, None, 0)) - spikes0
    ms_all, units_all = reduce_over_ranks(ms, units_per_step * args.steps, world, dev)

    # ---- the other launch granularity, for the record (not the headline)
    other = {"stream": "fused", "fused": "stream"}[args.mode]
    other_res = None
    if not args.no_other:
        g.set_option(B.ARB_OPT_FUSED_STEPS, fused_steps[other])
        _, t_now = timed_epochs(torch, g, t_now, 1, sync_all)
        oms, t_now = timed_epochs(torch, g, t_now, max(2, args.steps // 2), sync_all)
        n_o = max(2, args.steps // 2)
        oms_all, ounits_all = reduce_over_ranks(oms, units_per_step * n_o, world, dev)
        other_res = {"mode": other, "value": ounits_all / (oms_all * 1e-3), "unit": UNIT, "steps": n_o,
                     "ms_per_step": oms_all / n_o}
        g.set_option(B.ARB_OPT_FUSED_STEPS, fused_steps[args.mode])

    # ---- end to end through the C ABI with HOST buffers: every step uploads the state it starts
    # from (arb_set_state: V and synaptic conductances, pinned host memory), integrates one epoch,
    # and reads voltages and spikes back (arb_voltage, arb_spikes)
    n_e2e = max(2, min(args.steps, 4))
    hv = torch.empty(n_cv, dtype=torch.float64).pin_memory()
    hg = torch.empty(m["n_syn"], dtype=torch.float64).pin_memory()
    hv_np, hg_np = hv.numpy(), hg.numpy()
    g.voltage(out=hv_np)
    hg_np[:] = g.syn_g()
    sync_all()
    t0 = time.perf_counter()
    d2h_spikes = 0
    for _ in range(n_e2e):
        g.set_state(v=hv_np, syn_g=hg_np)
        t_now += EPOCH_MS
        g.advance(t_now, DT)
        g.voltage(out=hv_np)
        sc, st = g.spikes()
        d2h_spikes = 12 * len(sc)
    torch.cuda.synchronize()
    e2e_ms = (time.perf_counter() - t0) * 1e3
    e2e_ms_all, e2e_units = reduce_over_ranks(e2e_ms, units_per_step * n_e2e, world, dev)
    e2e = {"value": e2e_units / (e2e_ms_all * 1e-3), "unit": UNIT, "steps": n_e2e,
           "h2d_bytes_per_step": 8 * (n_cv + m["n_syn"]), "d2h_bytes_per_step": 8 * n_cv + d2h_spikes,
           "what": "arb_set_state(V, g from pinned host) + arb_advance(one epoch) + arb_voltage + arb_spikes to host; wall clock"}

    g.close()
    del g
    torch.cuda.empty_cache()

    # ---- configs[3] exactly as BASELINE.json words it (no external drive: the network stays silent);
    # the headline above adds the Poisson drive of SURVEY.md 8(d) C3(i), which costs event-split sub-steps
    as_written = None
    if not args.no_as_written:
        mu = W.config3(n_cells=args.cells, first_cell=rank * args.cells, driven=False)
        gu = B.Model(mu, device="cuda:%d" % local)
        gu.set_option(B.ARB_OPT_FUSED_STEPS, fused_steps[args.mode])
        tu = 0.0
        _, tu = timed_epochs(torch, gu, tu, 2, sync_all)
        gu.set_option(B.ARB_OPT_TIMING, 1)
        n_u = max(2, args.steps // 2)
        ums, tu = timed_epochs(torch, gu, tu, n_u, sync_all)
        utim = gu.timing()
        ums_all, uunits_all = reduce_over_ranks(ums, mu["n_cv"] * STEPS_PER_EPOCH * n_u, world, dev)
        spl = STEPS_PER_EPOCH if args.mode == "fused" else 1
        u_launch_ms = utim["cable_ms"] / max(1, utim["cable_launches"])
        u_ach = algorithmic_bytes_per_grid_step(mu) * spl / (u_launch_ms * 1e-3) / 1e9
        as_written = {"workload": "configs[3] as written (undriven, no events)", "value": uunits_all / (ums_all * 1e-3),
                      "unit": UNIT, "steps": n_u, "ms_per_step": ums_all / n_u, "avg_launch_ms": u_launch_ms,
                      "achieved_gbs": u_ach, "roofline_frac": u_ach / measured_peak_hbm()[0]}
        gu.close()
        del gu

    if rank != 0:
        return

    # ---- roofline of the dominant kernel (cable_group_kernel: every cell of C3 is in a cell group), measured
    # live with CUDA events on the model's stream
    peak, peak_src = measured_peak_hbm()
    steps_per_launch = STEPS_PER_EPOCH if args.mode == "fused" else 1
    alg = algorithmic_bytes_per_grid_step(m) * steps_per_launch
    avg_launch_ms = tim["cable_ms"] / max(1, tim["cable_launches"])
    achieved = alg / (avg_launch_ms * 1e-3) / 1e9 if avg_launch_ms > 0 else 0.0
    roofline = {"kernel": "cable_group_kernel", "bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s",
                "frac": achieved / peak, "traffic": committed_traffic("cable_group_kernel:" + args.mode),
                "peak_source": peak_src, "algorithmic_bytes_per_launch": alg,
                "avg_launch_ms": avg_launch_ms, "launches_timed": tim["cable_launches"],
                "kernel_share_of_step": tim["cable_ms"] / ms if ms > 0 else None,
                "epoch_boundary_ms_per_step": tim["event_ms"] / args.steps}
    # secondary (arithmetic) bound: DP instructions of a launch (committed ncu count) over the
    # fp64 rate measured live by the library's DFMA kernel
    try:
        dfma_rate, _ = B.arb_fp64_peak(torch.cuda.current_stream().cuda_stream)
        dp_inst = committed_traffic("cable_group_kernel:%s:dp_inst" % args.mode)
        roofline["fp64"] = {"peak_dfma_per_s": dfma_rate, "peak_source": "arb_fp64_peak (live DFMA microbenchmark)",
                            "dp_inst_per_launch": dp_inst,
                            "fp64_ms": (dp_inst / dfma_rate * 1e3) if dp_inst else None,
                            "hbm_ms": alg / (peak * 1e9) * 1e3,
                            "note": "roofline time = max(hbm_ms, fp64_ms): HBM-bound"}
    except Exception as e:  # the figure is context; the HBM roofline above is the claim
        roofline["fp64"] = {"error": str(e)}
    if args.mode == "fused":
        roofline["note"] = ("fused launches keep state on chip for 200 steps; algorithmic bytes are the level-A "
                            "per-step figure x 200, so frac > 1 means HBM traffic was avoided, not that work was skipped")

    cpu = None
    if not args.no_cpu_baseline:
        r = time_oracle(args.ref_cells, 2, 1)
        cpu = {"value": r["value"], "unit": UNIT, "cores": r["cores"], "kind": "oracle", "sample": r["sample"]}
        r1 = time_oracle(max(1, args.ref_cells // 10), 1, 1, threads=1)   # SURVEY.md 8(d) oracle timing (i)
        cpu["single_thread"] = {"value": r1["value"], "unit": UNIT, "cores": 1, "sample": r1["sample"]}

    line = {"metric": METRIC, "value": units_all / (ms_all * 1e-3), "unit": UNIT, "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_all / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic",
            "config": {"workload": "configs[3] C3 large: %d cells x 505 CVs (%d CVs), 50 expsyn + 50 connections/cell, "
                                   "200 Hz/cell Poisson drive, dt 0.025 ms; step = one 5 ms epoch (200 grid steps)"
                                   % (args.cells, n_cv),
                       "mode": args.mode, "cells_per_gpu": args.cells, "parallelism": "cells sharded, no collective",
                       "l2": "no flush needed: each grid step streams %.2f GB >> 126 MB L2" % (alg / steps_per_launch / 1e9),
                       "seed": int(W.BASE_SEED + 3)},
            "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches),
            "roofline": roofline, "cpu_baseline": cpu,
            "spikes": n_spikes, "spikes_per_s": n_spikes / (ms * 1e-3),
            "events_delivered": int(n_events), "events_per_s": n_events / (ms * 1e-3),
            "substep_overhead": float((sub1[1] - sub0[1]) / (m["n_cells"] * (sub1[0] - sub0[0])) - 1.0)}
    if other_res:
        line["fused_epoch" if other == "fused" else "stream"] = other_res
    if as_written:
        line["as_written"] = as_written
    print(json.dumps(line), flush=True)
    if world > 1:
        torch.distributed.destroy_process_group()


def selftest_dist():
    """CPU check of the N > 1 reduction (tests/test_bench_dist.py): gloo, fake per-rank figures."""
    import torch
    import torch.distributed as dist
    rank, world, _ = dist_env()
    dist.init_process_group("gloo")
    ms, units = reduce_over_ranks(10.0 * (rank + 1), 1000.0 * (rank + 1), world, torch.device("cpu"))
    dist.barrier()
    if rank == 0:
        print(json.dumps({"selftest": True, "n_gpus": world, "ms": ms, "units": units,
                          "value": units / (ms * 1e-3)}), flush=True)
    dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=8)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--mode", default="stream", choices=["stream", "fused"])
    ap.add_argument("--cells", type=int, default=100000, help="cells per GPU (configs[3]: 100000)")
    ap.add_argument("--ref-cells", type=int, default=2000, help="cells in the oracle's bounded sample")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-other", action="store_true", help="skip the other launch granularity")
    ap.add_argument("--no-as-written", action="store_true", help="skip the undriven (as worded in BASELINE.json) variant")
    ap.add_argument("--selftest-dist", action="store_true", help=argparse.SUPPRESS)
    args = ap.parse_args()
    if args.selftest_dist:
        return selftest_dist()
    if args.impl == "reference":
        return run_reference(args)
    if args.warmup < 3:
        print("note: fewer than 3 warm-up steps requested", file=sys.stderr)
    run_ours(args)


if __name__ == "__main__":
    main()
