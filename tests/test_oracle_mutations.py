"""Mutation check of the oracle's pins: each single-line mutation of a COPY of oracle/arb_oracle.c
must turn at least one pin of tests/test_oracle_pins.py red.  A mutation that survives marks a part
of the oracle as "parity unpinned".  The copies are built in a temporary directory and loaded through
ORC_MUTANT_LIB (oracle/orc.py); oracle/ itself is never modified.

The mutation list (what is changed, which pin is expected to catch it, the passage it pins):
  syn_half        I += 0.5 g (V - e)                 P13   PAPER.md:127-131 eq 2a, R7
  syn_sign        I += g (V + e)                     P13   R7 (reversal potential)
  gates_old_v     gate rates from V(t), not V'       P14   PAPER.md:148 "integrated with the updated voltage"
  clamp_window    t0 < t <= t1                       P15   R8
  hh_m2           m^3 -> m^2                         P9    R5
  area_scale      1e-2 -> 1.1e-2 (HH current)        P9    R2
  syn_decay       exp(-delta/tau) -> exp(-delta/(2 tau))   P8    R7
  spike_interp    no interpolation inside the step   P11   R10
  hines_parent    elimination updates the wrong row  P1
  assemble_diag   parent loses the child's sigma     P1/P2 PAPER.md:154
  delay_half      event time = spike + delay/2       P11
  weight_drop     g = w instead of g += w            P8    PAPER.md:150, R7
  lif_refractory  LIF: events are not ignored during t_ref             K1     R20
  lif_reset       LIF: reset to E_L instead of E_R                     K1     R20
  src_schedule    spike source: a spike at the interval's end emitted early (K2 compares exact times / counts)  K2  R20
  lin_syn_diag    linearised step: synaptic g missing on the diagonal   L1/L3  PAPER.md:152-156 (NEXT-2)
  lin_clamp_sign  linearised step: clamp current with the wrong sign   L1/L3  R8
  lin_hh_h        linearised step: g_Na without h                      L1/L4  R5
"""
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
SRC = os.path.join(ROOT, "oracle", "arb_oracle.c")
CFLAGS = ["-O2", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-fPIC", "-shared", "-std=c11"]

MUTATIONS = {
    "syn_half": ("I[i] += M->g[gs] * (v[i] - M->syn_e[gs]);", "I[i] += 0.5 * M->g[gs] * (v[i] - M->syn_e[gs]);", "p13"),
    "syn_sign": ("I[i] += M->g[gs] * (v[i] - M->syn_e[gs]);", "I[i] += M->g[gs] * (v[i] + M->syn_e[gs]);", "p13"),
    "gates_old_v": ("  c->v_prev = v[c->det];\n  for (int64_t i = 0; i < c->n; ++i) v[i] = x[i];",
                    "  c->v_prev = v[c->det];\n  double* vold = (double*)malloc((size_t)c->n * 8); memcpy(vold, v, (size_t)c->n * 8);\n"
                    "  for (int64_t i = 0; i < c->n; ++i) v[i] = x[i];", "p14"),
    "clamp_window": ("if (M->cl_t0[ck] <= t && t < M->cl_t1[ck]) I[", "if (M->cl_t0[ck] < t && t <= M->cl_t1[ck]) I[", "p15"),
    "hh_m2": ("double dens = M->gna[gi] * m * m * m * h", "double dens = M->gna[gi] * m * m * h", "p9"),
    "area_scale": ("I[i] += dens * M->area[gi] * 1e-2;", "I[i] += dens * M->area[gi] * 1.1e-2;", "p9"),
    "syn_decay": ("M->g[gs] = M->g[gs] * exp(-delta / M->syn_tau[gs]);", "M->g[gs] = M->g[gs] * exp(-delta / (2.0 * M->syn_tau[gs]));", "p8"),
    "spike_interp": ("c->new_spikes[c->n_new++] = t + delta * (M->theta - c->v_prev) / (vd - c->v_prev);",
                     "c->new_spikes[c->n_new++] = t + delta;", "p11"),
    "hines_parent": ("rhs[parent[i]] -= f * rhs[i];", "rhs[parent[i]] -= f * rhs[parent[i]];", "p1"),
    "assemble_diag": ("    d[parent[i]] += sigma;\n", "", "p1 or p2"),
    "delay_half": ("event e = { ts + M->conn_delay[kk],", "event e = { ts + 0.5 * M->conn_delay[kk],", "p11"),
    "lin_syn_diag": ("    gsum[i] += M->g[gs];\n", "", "l1 or l3"),
    "lin_clamp_sign": ("src[M->cl_cv[ck]] += M->cl_amp[ck];", "src[M->cl_cv[ck]] -= M->cl_amp[ck];", "l1 or l3"),
    "lin_hh_h": ("double gna = M->gna[gi] * m * m * m * h * sc,", "double gna = M->gna[gi] * m * m * m * sc,", "l1 or l4"),
    "lif_refractory": ("    if (te < c->t_ref_end) continue;", "", "k1"),
    "lif_reset": ("      v[0] = M->lif_e_r[ci];\n", "      v[0] = M->lif_e_l[ci];\n", "k1"),
    "src_schedule": ("M->src_time[c->src_cur] < tb) {", "M->src_time[c->src_cur] <= tb) {", "k2"),
    "weight_drop": ("M->g[c->syn0 + c->q[c->qh].syn] += c->q[c->qh].w;", "M->g[c->syn0 + c->q[c->qh].syn] = c->q[c->qh].w;", "p8"),
}
# gates_old_v needs a second edit: the rate call reads the saved copy
EXTRA = {"gates_old_v": ("orc_hh_rates(v[i], r);\n    double* st[3]", "orc_hh_rates(vold[i], r);\n    double* st[3]")}


def _pins(lib, expr):
    env = dict(os.environ)
    if lib:
        env["ORC_MUTANT_LIB"] = lib
    else:
        env.pop("ORC_MUTANT_LIB", None)
    return subprocess.run([sys.executable, "-m", "pytest", os.path.join(ROOT, "tests", "test_oracle_pins.py"), "-x", "-q",
                           "-k", expr, "-p", "no:cacheprovider"], cwd=ROOT, env=env, capture_output=True, text=True, timeout=120)


@pytest.mark.parametrize("name", sorted(MUTATIONS))
def test_mutation_is_caught(tmp_path, name):
    old, new, pins = MUTATIONS[name]
    src = open(SRC).read()
    assert src.count(old) == 1, "mutation target not found exactly once: " + name
    src = src.replace(old, new)
    if name in EXTRA:
        assert src.count(EXTRA[name][0]) == 1
        src = src.replace(*EXTRA[name])
    c = tmp_path / "arb_oracle.c"
    c.write_text(src)
    lib = str(tmp_path / "liborc_mutant.so")
    subprocess.check_call(["gcc", *CFLAGS, "-I", os.path.join(ROOT, "oracle"), "-o", lib, str(c), "-lm"])
    r = _pins(lib, pins)
    assert r.returncode != 0 and " failed" in r.stdout, "mutation %s survived the pins %s:\n%s" % (name, pins, r.stdout[-1500:])


def test_unmutated_oracle_passes_the_same_pins():
    r = _pins(None, "p1 or p2 or p8 or p9 or p11 or p13 or p14 or p15 or l1 or l3 or l4 or k1 or k2")
    assert r.returncode == 0, r.stdout[-2000:]
