"""The paper's own ring-network cell (~130 control volumes, 10,000 exponential synapses
per cell, one of them wired) through the C ABI: cable-step time per grid step with one launch per
step ("stream") and with whole epochs per launch ("fused"), as one JSON line.

    python -m paper_1901_07454_b200.examples.paper_ring [n_cells]

SURVEY.md 8(f) NEXT-1 workload; not the bench.py headline.  Needs a B200 and the built library."""
import json
import sys

from paper_1901_07454_b200 import binding as B, workloads as W

DT, EPOCH_MS = 0.025, 5.0


def main(n_cells=2048):
    m = W.paper_ring(n_cells=n_cells, t_end=40.0)
    g = B.Model(m)
    st = g.stats()
    # level-A algorithmic bytes per grid step: 48 B per CV, 80 B per HH CV (the soma), 20 B per synapse
    alg = 48 * m["n_cv"] + 80 * n_cells + 20 * m["n_syn"]
    out = {"workload": "paper ring cell", "n_cells": n_cells, "n_cv": int(m["n_cv"]), "n_syn": int(m["n_syn"]),
           "units": st["units"], "groups": st["groups"], "algorithmic_bytes_per_grid_step": alg}
    t = 0.0
    for mode, fused in (("stream", 1), ("fused", 0)):
        g.set_option(B.ARB_OPT_FUSED_STEPS, fused)
        t += EPOCH_MS
        g.advance(t, DT)                       # warm-up epoch
        g.set_option(B.ARB_OPT_TIMING, 1)
        t += EPOCH_MS
        g.advance(t, DT)
        tim = g.timing()
        g.set_option(B.ARB_OPT_TIMING, 0)
        ms = tim["cable_ms"] / round(EPOCH_MS / DT)
        out[mode] = {"cable_ms_per_grid_step": ms, "synapse_steps_per_s": m["n_syn"] / (ms * 1e-3),
                     "algorithmic_gb_per_s": alg / (ms * 1e-3) / 1e9}
    out["spikes"] = int(len(g.spikes()[0]))
    g.close()
    print(json.dumps(out), flush=True)


if __name__ == "__main__":
    main(int(sys.argv[1]) if len(sys.argv) > 1 else 2048)
