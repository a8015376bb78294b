#!/usr/bin/env python
"""bench.py - throughput of the cable-step hot path on B200.

    python bench.py [--config 0|1|2|3|4|ring] [--gpus N] [--steps K] [--warmup W]
                    [--impl ours|reference] [--mode stream|fused] [--step linearised]

Workloads (seeded, synthetic: paper_1901_07454_b200.workloads; they stand in for the paper's ring and
random-connectivity benchmark networks):
  --config 3 (default, the headline)  BASELINE.json configs[3] "C3 large": 100,000 cells, depth-6 trees of
             63 branches x 8 control volumes (~5.05e7 CVs), 50 exponential synapses and 50 incoming
             connections per cell, dt = 0.025 ms, 200 Hz/cell Poisson drive; the
             network exactly as BASELINE.json words it (no drive) is measured in the same run ("as_written")
  --config 0 / 1 / 2 / 4              the other BASELINE.json configs at their full sizes
  --config ring                       the paper's own ring cell (~130 CVs and 10,000
                                      exponential synapses per cell), 2,048 cells

A bench "step" is ONE EPOCH of the network as the library runs it (`epoch_steps` grid steps of dt: the
minimum connection delay; 1,024 steps where there are no connections): event delivery,
mechanism currents, matrix assembly, Hines solve, voltage update, state update and threshold test once per
grid step (rows a0..a6 of SURVEY.md 8(a)), then the epoch boundary that turns the epoch's spikes into
queued events (row a7).  metric = compartment-steps/s = (number of CVs) x (grid steps) / device time of
arb_advance.

mode "stream" (default, the headline): one cable-step launch per grid step, every cell's state and
coefficients stream through HBM each step - the configuration SURVEY.md 8(d) defines the level-A HBM
roofline for.  mode "fused": the same kernels keep a cell's state on chip for a whole epoch
(ARB_OPT_FUSED_STEPS = 0); reported beside the headline under "fused_epoch".

N > 1 (torchrun): every rank integrates its own closed network of the same population (weak scaling, no
data-path collective); value = CV-steps of all ranks / max-over-ranks device time.

--impl reference: times the CPU oracle (oracle/, plain fp64 C, as it stands) on this box's host cores on
a bounded sample of the same workload; rank 0 only.
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

UNIT = "CV-steps/s"
DT = 0.025
FALLBACK_HBM_GBS = 6650.0   # /opt/skills/guides/B200_PROFILING.md fallback
NOMINAL_HBM_GBS = 8000.0    # BASELINE.json north_star "~8 TB/s"


# --------------------------------------------------------------------------------------------
# workloads
# --------------------------------------------------------------------------------------------
class Workload:
    """What `--config` selects: how to build the network for `ms` of simulated time and how to cut a
    bounded sample for the oracle."""

    def __init__(self, key, label, make, ref_cells, full_cells):
        self.key, self.label, self.make, self.ref_cells, self.full_cells = key, label, make, ref_cells, full_cells


def _workloads():
    from paper_1901_07454_b200 import workloads as W
    return {
        "0": Workload("0", "configs[0] C0 single cell: HH soma + 10-CV passive dendrite, 0.1 nA clamp 10-60 ms",
                      lambda n, ms, first, driven: W.config0(), 1, 1),
        "1": Workload("1", "configs[1] C1 ring: %d cells x 301 CVs, 10 expsyn, ring delay 5 ms, weight 0.01 uS (synapse 0 on the soma, DESIGN.md R19)",
                      lambda n, ms, first, driven: W.config1(n_cells=n, t_end=ms, ring_syn_on_soma=driven), 1000, 1000),
        "2": Workload("2", "configs[2] C2 random: %d cells x 301 CVs, 100 connections + 20 Poisson (10 Hz) synapses per cell",
                      lambda n, ms, first, driven: W.config2(n_cells=n, t_end=ms), 2000, 10000),
        "3": Workload("3", "configs[3] C3 large: %d cells x 505 CVs, 50 expsyn + 50 connections/cell, 200 Hz/cell Poisson drive",
                      lambda n, ms, first, driven: W.config3(n_cells=n, t_end=ms, driven=driven, first_cell=first), 2000, 100000),
        "4": Workload("4", "configs[4] C4 heterogeneous: %d cells, depth U{2..8}, 4..40 CVs/branch, HH on soma + 10%% of dendritic CVs, 30 connections/cell, 200 Hz/cell Poisson drive",
                      lambda n, ms, first, driven: W.config4(n_cells=n, t_end=ms), 2000, 50000),
        "ring": Workload("ring", "paper ring cell (PAPER.md:289): %d cells x ~130 CVs x 10,000 expsyn, one wired (SURVEY.md 8(f) NEXT-1)",
                         lambda n, ms, first, driven: W.paper_ring(n_cells=n, t_end=ms), 64, 2048),
    }


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


def algorithmic_bytes_per_grid_step(m, linearised=False):
    """Level-A bytes one grid step must move:
    48 B per CV (V read + write, rhs coefficients a,b, solver factors f, 1/d), 4 B per branch
    (parent link), 80 B per HH CV (m,h,n read + write, three conductances, slot), 20 B per synapse
    (g read + write, CV index).  The conductance-linearised step re-assembles
    and re-eliminates every step: C/dt, sum(sigma) + G, sigma, G e instead of a, b, f, 1/d = the same
    48 B per CV as implemented here (SURVEY's 56-60 B counts u separately from sigma)."""
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
    return 48 * m["n_cv"] + 4 * n_branch + 80 * n_hh + 20 * synapse_instances(m)


def synapse_instances(m):
    """Synapse instances a step integrates: one per synapse, except in cells with >= 1,024 synapses, where the library
    keeps ONE conductance per run of synapses on the same control volume with the same (tau, e) (R22;
    SURVEY.md 8(f) NEXT-1, second half) - the roofline is then quoted against that smaller count."""
    so = np.asarray(m["syn_off"], np.int64)
    per_cell = np.diff(so)
    big = np.flatnonzero(per_cell >= 1024)
    n = int(m["n_syn"])
    for c in big:
        a, b = int(so[c]), int(so[c + 1])
        key = np.stack([m["syn_cv"][a:b].astype(np.float64), m["syn_tau"][a:b], m["syn_e"][a:b]], axis=1)
        runs = len(np.unique(key, axis=0))
        if 2 * runs <= b - a:
            n -= (b - a) - runs
    return n


def committed_traffic(key):
    """(value, source) of row `key` of profiles/roofline_traffic.csv: figures copied from committed ncu
    captures (the capture and its command are named in the row), or (None, None)."""
    p = os.path.join(ROOT, "profiles", "roofline_traffic.csv")
    try:
        with open(p) as f:
            for line in f:
                c = [x.strip() for x in line.split(",", 3)]
                if len(c) >= 3 and c[0] == key:
                    return float(c[2]), (c[3] if len(c) > 3 else None)
    except Exception:
        pass
    return None, None


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


def epoch_steps_of(m):
    """Grid steps of one epoch as the library cuts them (include/arbb200.h, arb_advance)."""
    if m["n_conn"] == 0:
        return 1024
    return max(1, min(1024, int(np.floor(float(np.min(m["conn_delay"])) / m["dt"] - 1e-6))))


# --------------------------------------------------------------------------------------------
# reference arm / cpu_baseline: the oracle on the host cores
# --------------------------------------------------------------------------------------------
def oracle_sample(wl, n_cells_sample, ms):
    """First `n_cells_sample` cells of the population as an isolated network (their external events
    and clamps kept, connections dropped): the same per-cell work as in the full network."""
    from paper_1901_07454_b200 import workloads as W
    if wl.full_cells == 1:
        return wl.make(1, ms, 0, True)
    m = wl.make(n_cells_sample + 1, ms, 0, True)
    return W.take_cells(m, np.arange(n_cells_sample))


def time_oracle(wl, sample_cells, steps, warmup, epoch_steps, threads=None, linearised=False):
    from oracle import orc
    orc.build()
    cores = threads or os.cpu_count() or 1
    ms = (warmup + steps + 1) * epoch_steps * DT
    sub = oracle_sample(wl, sample_cells, ms)
    o = orc.Oracle(sub, threads=cores)
    if linearised:
        o.set_linearised(True)
    t = 0.0
    times = []
    for i in range(warmup + steps):
        t0 = time.perf_counter()
        t += epoch_steps * DT
        o.advance(t, DT)
        dt_ = time.perf_counter() - t0
        if i >= warmup:
            times.append(dt_)
    o.close()
    per_step = float(np.mean(times))
    return dict(value=sub["n_cv"] * epoch_steps / per_step, ms_per_step=per_step * 1e3, cores=cores,
                sample="first %d cells of %s (%d CVs, connections dropped, external events kept), "
                       "%d epochs of %d steps, %s" % (sub["n_cells"], wl.key if wl.key == "ring" else "C" + wl.key, sub["n_cv"], steps,
                                                      epoch_steps, "OpenMP over cells" if cores > 1 else "one thread"))


def metric_name(wl, linearised):
    return "compartment-steps/sec (fp64), %s%s" % ("C" + wl.key if wl.key != "ring" else "paper ring cell",
                                                   ", conductance-linearised step" if linearised else "")


def run_reference(args):
    rank, world, _ = dist_env()
    if rank != 0:
        return
    wl = _workloads()[args.config]
    cells = args.cells or wl.full_cells
    probe = wl.make(min(cells, 8) if wl.full_cells > 1 else 1, 10.0, 0, True)
    es = epoch_steps_of(probe)
    ref_cells = min(args.ref_cells or wl.ref_cells, cells)
    lin = args.step == "linearised"
    r = time_oracle(wl, ref_cells, args.steps, min(args.warmup, 1), es, linearised=lin)
    line = {"impl": "reference", "metric": metric_name(wl, lin), "value": r["value"], "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": min(args.warmup, 1), "ms_per_step": r["ms_per_step"],
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic",
            "config": {"workload": (wl.label % cells if "%d" in wl.label else wl.label) + " (bounded sample: %s)" % r["sample"]},
            "cpu_baseline": {"value": r["value"], "unit": UNIT, "cores": r["cores"], "kind": "oracle",
                             "sample": r["sample"]},
            "e2e": {"value": r["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# --------------------------------------------------------------------------------------------
# our arm
# --------------------------------------------------------------------------------------------
def timed_epochs(torch, g, t_now, n, step_ms, sync_all):
    """n epochs through arb_advance, device time by CUDA events on the model's stream (one event per
    epoch boundary: total and per-epoch times)."""
    sync_all()
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(n + 1)]
    ev[0].record(g.stream)
    for i in range(n):
        t_now += step_ms
        g.advance(t_now, DT)
        ev[i + 1].record(g.stream)
    torch.cuda.synchronize()
    ms = ev[0].elapsed_time(ev[n]) if n else 0.0
    per = [ev[i].elapsed_time(ev[i + 1]) for i in range(n)]
    sync_all()
    return ms, per, t_now


def run_ours(args):
    import torch
    rank, world, local = dist_env()
    if args.gpus != world:
        raise SystemExit("bench.py: --gpus %d but WORLD_SIZE is %d: for N > 1 launch with `python -m torch.distributed.run "
                         "--nnodes=1 --nproc-per-node N --master-addr 127.0.0.1 bench.py --gpus N ...`" % (args.gpus, world))
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
    for kv in args.layout:
        k, v = kv.split("=")
        assert k in B.OPTION_FIELDS, k
        B.LAYOUT_DEFAULTS[k] = int(v)
    wl = _workloads()[args.config]
    cells = args.cells or wl.full_cells
    lin = args.step == "linearised"
    # simulated time the run needs: every timed leg advances the same model
    probe = wl.make(min(cells, 8) if wl.full_cells > 1 else 1, 10.0, 0, True)
    es = epoch_steps_of(probe)
    step_ms = es * DT
    n_other = 0 if args.no_other else 1 + max(2, args.steps // 2)
    n_e2e = max(2, min(args.steps, 4))
    total_ms = (args.warmup + args.steps + n_other + n_e2e + 2) * step_ms
    sm = None
    if args.exchange:
        if args.config != "3":
            raise SystemExit("bench.py --exchange is implemented for --config 3")
        from paper_1901_07454_b200 import sharded as S
        m = W.config3(n_cells=cells, t_end=total_ms, first_cell=rank * cells, n_global=world * cells)
        sm = S.ShardedModel(B, None, rank, world, S.DistGroup(torch, dev) if world > 1 else None, device="cuda:%d" % local, local=m)
        g = sm.model
    else:
        m = wl.make(cells, total_ms, rank * cells, True)
        g = B.Model(m, device="cuda:%d" % local)
    assert epoch_steps_of(m) == es
    if sm is not None:           # every epoch: integrate, then exchange the epoch's spikes (inside the timed region)
        _adv = g.advance
        def _advance_and_exchange(t, dt):
            if args.overlap:             # half-epoch exchange intervals, the all-gather hidden behind the next half-epoch
                g.advance = _adv         # (the sharded loop calls the model's own advance)
                try:
                    sm.t = g.time()
                    sm.advance(t, dt)
                finally:
                    g.advance = _advance_and_exchange
                return
            _adv(t, dt)
            sm.exchange()
        g.advance = _advance_and_exchange
        sm.overlap = bool(args.overlap)
    fused_steps = {"stream": 1, "fused": 0}
    g.set_option(B.ARB_OPT_FUSED_STEPS, fused_steps[args.mode])
    if lin:
        g.set_option(B.ARB_OPT_LINEARISED, 1)
    n_cv = m["n_cv"]
    units_per_step = n_cv * es

    # ---- device-resident timing: W warm-up epochs, K timed epochs
    t_now = 0.0
    _, _, t_now = timed_epochs(torch, g, t_now, args.warmup, step_ms, sync_all)
    g.set_option(B.ARB_OPT_TIMING, 1)
    st0 = g.stats()
    l0 = st0["launches"]
    sub0 = g.probe(B.ARB_PROBE_NSTEPS)
    spikes0 = int(B.lib().arb_spikes(g._h, None, None, 0))
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    ms, per_step, t_now = timed_epochs(torch, g, t_now, args.steps, step_ms, sync_all)
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
        _, _, t_now = timed_epochs(torch, g, t_now, 1, step_ms, sync_all)
        n_o = max(2, args.steps // 2)
        oms, _, t_now = timed_epochs(torch, g, t_now, n_o, step_ms, sync_all)
        oms_all, ounits_all = reduce_over_ranks(oms, units_per_step * n_o, world, dev)
        other_res = {"mode": other, "value": ounits_all / (oms_all * 1e-3), "unit": UNIT, "steps": n_o,
                     "ms_per_step": oms_all / n_o}
        g.set_option(B.ARB_OPT_FUSED_STEPS, fused_steps[args.mode])

    # ---- end to end through the C ABI with HOST buffers: every step uploads the state it starts
    # from (arb_set_state: V and synaptic conductances, pinned host memory), integrates one epoch,
    # and reads voltages and the epoch's spikes back (arb_voltage, arb_spikes, arb_clear_spikes)
    hv = torch.empty(n_cv, dtype=torch.float64).pin_memory()
    hg = torch.empty(max(1, m["n_syn"]), dtype=torch.float64).pin_memory()
    hv_np, hg_np = hv.numpy(), hg.numpy()[:m["n_syn"]]
    g.voltage(out=hv_np)
    hg_np[:] = g.syn_g()
    g.clear_spikes()
    sync_all()
    t0 = time.perf_counter()
    d2h_spikes = 0
    for _ in range(n_e2e):
        g.set_state(v=hv_np, syn_g=hg_np if m["n_syn"] else None)
        t_now += step_ms
        g.advance(t_now, DT)
        g.voltage(out=hv_np)
        sc, st = g.spikes()
        g.clear_spikes()
        d2h_spikes = max(d2h_spikes, 12 * len(sc))
    torch.cuda.synchronize()
    e2e_ms = (time.perf_counter() - t0) * 1e3
    e2e_ms_all, e2e_units = reduce_over_ranks(e2e_ms, units_per_step * n_e2e, world, dev)
    e2e = {"value": e2e_units / (e2e_ms_all * 1e-3), "unit": UNIT, "steps": n_e2e,
           "h2d_bytes_per_step": 8 * (n_cv + m["n_syn"]), "d2h_bytes_per_step": 8 * n_cv + d2h_spikes,
           "what": "arb_set_state(V, g from pinned host) + arb_advance(one epoch) + arb_voltage + arb_spikes + arb_clear_spikes to host; wall clock"}

    layout = {k: st1[k] for k in ("groups", "classes", "units", "warp_units", "forests")}
    g.close()
    del g
    torch.cuda.empty_cache()

    # ---- configs[3] exactly as BASELINE.json words it (no external drive: the network stays silent);
    # the headline above adds the Poisson drive of SURVEY.md 8(d) C3(i), which costs event-split sub-steps
    as_written = None
    if args.config in ("3", "1") and not args.no_as_written:    # C1: the ring synapse on a random dendritic CV (R19)
        mu = wl.make(cells, 10.0, rank * cells, False)
        gu = B.Model(mu, device="cuda:%d" % local)
        gu.set_option(B.ARB_OPT_FUSED_STEPS, fused_steps[args.mode])
        if lin:
            gu.set_option(B.ARB_OPT_LINEARISED, 1)
        tu = 0.0
        _, _, tu = timed_epochs(torch, gu, tu, 2, step_ms, sync_all)
        gu.set_option(B.ARB_OPT_TIMING, 1)
        n_u = max(2, args.steps // 2)
        ums, _, tu = timed_epochs(torch, gu, tu, n_u, step_ms, sync_all)
        utim = gu.timing()
        ums_all, uunits_all = reduce_over_ranks(ums, mu["n_cv"] * es * n_u, world, dev)
        u_step_ms = utim["cable_ms"] / max(1, n_u * es)
        u_ach = algorithmic_bytes_per_grid_step(mu, lin) / (u_step_ms * 1e-3) / 1e9
        as_written = {"workload": ("configs[3] as written (undriven, no events)" if args.config == "3" else
                                   "configs[1] as stated (ring synapse on a random dendritic compartment: the ring dies after the kicked cell, DESIGN.md R19)"),
                      "value": uunits_all / (ums_all * 1e-3),
                      "unit": UNIT, "steps": n_u, "ms_per_step": ums_all / n_u, "cable_ms_per_grid_step": u_step_ms,
                      "achieved_gbs": u_ach, "roofline_frac": u_ach / measured_peak_hbm()[0]}
        gu.close()
        del gu

    if rank != 0:
        return

    # ---- roofline of the cable step (the kernels launched once per grid step; for C1-C3 that is
    # cable_group_kernel alone), measured live with CUDA events on the model's stream
    peak, peak_src = measured_peak_hbm()
    alg_step = algorithmic_bytes_per_grid_step(m, lin)
    grid_steps_timed = args.steps * es
    cable_ms_per_grid_step = tim["cable_ms"] / grid_steps_timed
    launches_per_grid_step = tim["cable_launches"] / grid_steps_timed
    kernels = []
    if layout["groups"]:
        kernels.append("cable_group_kernel")
    if layout["forests"]:
        kernels.append("cable_forest_kernel")
    if layout["units"] - layout["forests"] > 0:
        kernels.append("cable_block_kernel")
    achieved = alg_step / (cable_ms_per_grid_step * 1e-3) / 1e9 if cable_ms_per_grid_step > 0 else 0.0
    tkey = "C%s:%s:%s" % (args.config, "+".join(kernels), args.mode) + (":linearised" if lin else "")
    traffic, traffic_src = committed_traffic(tkey)
    roofline = {"kernel": "+".join(kernels), "bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s",
                "frac": achieved / peak, "frac_nominal_8tbs": achieved / NOMINAL_HBM_GBS,
                "traffic": traffic, "traffic_source": traffic_src,
                "peak_source": peak_src, "algorithmic_bytes_per_grid_step": alg_step, "synapse_instances": synapse_instances(m), "synapses": int(m["n_syn"]),
                "frac_if_every_synapse_were_integrated": (alg_step + 20 * (int(m["n_syn"]) - synapse_instances(m))) / (cable_ms_per_grid_step * 1e-3) / 1e9 / peak if cable_ms_per_grid_step > 0 else 0.0,
                "cable_ms_per_grid_step": cable_ms_per_grid_step, "launches_per_grid_step": launches_per_grid_step,
                "launches_timed": tim["cable_launches"],
                "kernel_share_of_step": tim["cable_ms"] / ms if ms > 0 else None,
                "epoch_boundary_ms_per_step": tim["event_ms"] / args.steps,
                "what": "achieved = level-A algorithmic bytes of one grid step / device time of the cable-step launches of "
                        "one grid step (CUDA events on the model's stream around the launches of every epoch)"}
    if args.mode == "fused":
        roofline["note"] = ("fused launches keep state on chip for an epoch; algorithmic bytes are the level-A per-step "
                            "figure, so frac > 1 means HBM traffic was avoided, not that work was skipped")
    if alg_step < 126e6:
        roofline["l2_note"] = "the per-step working set (%.1f MB) fits the 126 MB L2: not an HBM-bound case, frac is context only" % (alg_step / 1e6)
    # secondary (arithmetic) bound: DP instructions of a grid step (committed ncu count) over the
    # fp64 rate measured live by the library's DFMA kernel
    try:
        dfma_rate, _ = B.arb_fp64_peak(torch.cuda.current_stream().cuda_stream)
        dp_inst, dp_src = committed_traffic(tkey + ":dp_inst")
        roofline["fp64"] = {"peak_dfma_per_s": dfma_rate, "peak_source": "arb_fp64_peak (live DFMA microbenchmark)",
                            "dp_inst_per_grid_step": dp_inst, "dp_inst_source": dp_src,
                            "fp64_ms": (dp_inst / dfma_rate * 1e3) if dp_inst else None,
                            "hbm_ms": alg_step / (peak * 1e9) * 1e3}
    except Exception as e:  # the figure is context; the HBM roofline above is the claim
        roofline["fp64"] = {"error": str(e)}

    cpu = None
    if not args.no_cpu_baseline:
        ref_cells = min(args.ref_cells or wl.ref_cells, cells)
        ref_steps = 2 if es * ref_cells * (n_cv / max(1, cells)) < 5e8 else 1
        r = time_oracle(wl, ref_cells, ref_steps, 1, es, linearised=lin)
        cpu = {"value": r["value"], "unit": UNIT, "cores": r["cores"], "kind": "oracle", "sample": r["sample"]}
        r1 = time_oracle(wl, max(1, ref_cells // 10), 1, 1, es, threads=1, linearised=lin)   # SURVEY.md 8(d) oracle timing (i)
        cpu["single_thread"] = {"value": r1["value"], "unit": UNIT, "cores": 1, "sample": r1["sample"]}

    label = wl.label % cells if "%d" in wl.label else wl.label
    line = {"metric": metric_name(wl, lin), "value": units_all / (ms_all * 1e-3), "unit": UNIT, "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_all / args.steps,
            "ms_per_step_median": float(np.median(per_step)), "value_median": units_per_step * world / (float(np.median(per_step)) * 1e-3),
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic",
            "config": {"workload": "%s (%d CVs), dt 0.025 ms; step = one epoch of %d grid steps" % (label, n_cv, es),
                       "mode": args.mode, "step_kind": args.step, "cells_per_gpu": cells,
                       "parallelism": (("one network, cells sharded by rank, spikes all-gathered every half epoch behind the next half-epoch's integration" if args.overlap else "one network, cells sharded by rank, spikes all-gathered once per epoch") if args.exchange
                                       else "cells sharded, no collective (one closed network per rank)"), "layout": layout, "layout_options": dict(B.LAYOUT_DEFAULTS),
                       "l2": ("no flush needed: each grid step streams %.2f GB >> 126 MB L2" % (alg_step / 1e9)) if alg_step > 4e8
                             else "working set of %.1f MB per grid step is L2-resident; no flush (every step rewrites the whole state)" % (alg_step / 1e6),
                       "seed": int(W.BASE_SEED + (5 if args.config == "ring" else int(args.config)))},
            "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches),
            "roofline": roofline, "cpu_baseline": cpu,
            "spikes": n_spikes, "spikes_per_s": n_spikes / (ms * 1e-3),
            "events_delivered": int(n_events), "events_per_s": n_events / (ms * 1e-3),
            "substep_overhead": float((sub1[1] - sub0[1]) / (m["n_cells"] * (sub1[0] - sub0[0])) - 1.0)}
    if m["n_syn"] > 10 * n_cv:
        line["synapse_steps_per_s"] = m["n_syn"] * es * args.steps * world / (ms_all * 1e-3)
    if other_res:
        line["fused_epoch" if other == "fused" else "stream"] = other_res
    if as_written:
        line["as_written"] = as_written
    print(json.dumps(line), flush=True)
    if world > 1:
        torch.distributed.destroy_process_group()


def selftest_dist():
    """CPU check of the N > 1 reduction (tests/test_bench_cpu.py): gloo, fake per-rank figures."""
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
    ap.add_argument("--config", default="3", choices=["0", "1", "2", "3", "4", "ring"])
    ap.add_argument("--mode", default="stream", choices=["stream", "fused"])
    ap.add_argument("--step", default="explicit", choices=["explicit", "linearised"],
                    help="explicit: membrane currents from V(t) (reading R1, the headline); linearised: membrane "
                         "conductances on the diagonal, matrix re-assembled and re-eliminated every step (SURVEY.md 8(f) NEXT-2)")
    ap.add_argument("--cells", type=int, default=0, help="cells per GPU (default: the config's full size)")
    ap.add_argument("--ref-cells", type=int, default=0, help="cells in the oracle's bounded sample")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-other", action="store_true", help="skip the other launch granularity")
    ap.add_argument("--no-as-written", action="store_true", help="skip the undriven (as worded in BASELINE.json) variant of C3")
    ap.add_argument("--exchange", action="store_true",
                    help="config 3, N > 1: the ranks share ONE network of N x cells cells (cells sharded, connections by destination "
                         "owner) and all-gather their spikes once per epoch (paper_1901_07454_b200/sharded.py, SURVEY.md 8(f) NEXT-3) "
                         "instead of integrating one closed network each")
    ap.add_argument("--overlap", action="store_true",
                    help="with --exchange: exchange every half epoch and hide the all-gather behind the next half-epoch's "
                         "integration (PAPER.md:96, 200)")
    ap.add_argument("--layout", action="append", default=[], metavar="KEY=VALUE",
                    help="arb_desc layout / capacity option, e.g. layout_forest_cv=2048 (default: the library's)")
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
