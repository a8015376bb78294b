"""Seeded synthetic input generators (INPUTS ONLY - none of the method's arithmetic lives here).

Both the CUDA library (through ``paper_1901_07454_b200.binding``) and the CPU oracle (through
``oracle/orc.py``) consume the plain ``dict`` of NumPy arrays these functions return.  The keys are
the fields of ``arb_desc`` (include/arbb200.h), i.e. the paper's problem statement: per-cell
control volumes (PAPER.md:121-146 - c_i, S_i, sigma_ij), mechanisms named at PAPER.md:289
(HH soma, passive dendrites, exponential synapses), connections as the 5-tuple of PAPER.md:96 and
spike detectors.

The five ``config(k)`` workloads are the shapes listed in BASELINE.json ``configs`` (they stand in
for the paper's ring and random-connectivity benchmark networks, which are not
published as data).  Recipe (also in DESIGN.md):

* RNG: every cell ``c`` of config ``k`` owns ``numpy.random.default_rng([190107454 + k, c])`` and
  draws, in this order: branch lengths, branch diameters, (C4: topology first), synapse sites,
  incoming-connection sources, delays, external (Poisson) events.  A prefix of cells therefore has
  the same morphologies whatever the network size.
* Geometry -> control volumes (reading R3 of SURVEY.md 8(c)): one CV per cylinder segment, node at
  its centre; soma is CV 0, a cylinder with L = d = sqrt(area/pi).  Axial resistance between two
  neighbouring centres is half of each segment's resistance, R[MOhm] = 1e-2 * 4 Ra L / (pi d^2).
* CV order: soma, then branches in breadth-first order, proximal -> distal inside a branch, so
  ``parent < index`` always holds.
"""
from __future__ import annotations

import math
import numpy as np

BASE_SEED = 190107454

# R5/R6 parameter values (BASELINE.json configs[0])
GNABAR, GKBAR, GL = 0.12, 0.036, 3e-4          # S/cm^2
ENA, EK, EL = 50.0, -77.0, -54.3                # mV
G_PAS, E_PAS = 1e-5, -65.0                      # S/cm^2, mV
CM, RA = 1.0, 100.0                             # uF/cm^2, Ohm*cm
SOMA_AREA = 500.0                               # um^2
SYN_TAU, SYN_E = 2.0, 0.0                       # ms, mV
THRESHOLD = -10.0                               # mV
DT = 0.025                                      # ms


# ----------------------------------------------------------------------------------------------
# geometry -> control volumes
# ----------------------------------------------------------------------------------------------
def seg_resistance(length_um, diam_um, ra=RA):
    """Axial resistance [MOhm] of a cylinder segment (units: SURVEY.md 8 'Units')."""
    return 1e-2 * 4.0 * ra * length_um / (math.pi * diam_um * diam_um)


def soma_dims(area=SOMA_AREA):
    d = math.sqrt(area / math.pi)
    return d, d  # L, d


def cell_cvs(branch_parent, branch_ncv, branch_len, branch_diam, soma_area=SOMA_AREA):
    """Control volumes of one cell.

    branch_parent[b] = parent branch (-1: attached to the soma); branches are given in an order
    where parent < child.  Returns (parent[int32], area, raxial, first_cv_of_branch).
    """
    nb = len(branch_parent)
    ncv = 1 + int(np.sum(branch_ncv))
    parent = np.empty(ncv, np.int32)
    area = np.empty(ncv)
    rax = np.empty(ncv)
    ls, ds = soma_dims(soma_area)
    parent[0], area[0], rax[0] = -1, soma_area, 1.0   # root raxial is ignored by the library
    half_soma = 0.5 * seg_resistance(ls, ds)
    first = np.empty(nb, np.int64)
    last = np.empty(nb, np.int64)
    half = np.empty(nb)
    pos = 1
    for b in range(nb):
        n = int(branch_ncv[b])
        seg_l = branch_len[b] / n
        r = seg_resistance(seg_l, branch_diam[b])
        half[b] = 0.5 * r
        first[b], last[b] = pos, pos + n - 1
        idx = np.arange(pos, pos + n)
        parent[idx] = idx - 1
        area[idx] = math.pi * branch_diam[b] * seg_l
        rax[idx] = r
        pb = int(branch_parent[b])
        if pb < 0:
            parent[pos] = 0
            rax[pos] = half_soma + half[b]
        else:
            parent[pos] = last[pb]
            rax[pos] = half[pb] + half[b]
        pos += n
    return parent, area, rax, first


def _uniform_topology_cvs(bp, n, L, D):
    """Vectorised ``cell_cvs`` for N cells sharing one topology (bp) and n CVs per branch.

    L, D: [N, nb].  Returns parent[ncv] (shared), area[N, ncv], rax[N, ncv].
    """
    N, nb = L.shape
    ncv = 1 + nb * n
    parent = np.arange(-1, ncv - 1, dtype=np.int32)
    for b in range(nb):
        parent[1 + b * n] = 0 if bp[b] < 0 else (bp[b] + 1) * n
    seg_l = L / n
    r = 1e-2 * 4.0 * RA * seg_l / (math.pi * D * D)          # [N, nb]
    a = math.pi * D * seg_l
    area = np.empty((N, ncv))
    rax = np.empty((N, ncv))
    area[:, 0] = SOMA_AREA
    rax[:, 0] = 1.0
    area[:, 1:] = np.repeat(a, n, axis=1)
    rax[:, 1:] = np.repeat(r, n, axis=1)
    ls, ds = soma_dims()
    half_soma = 0.5 * seg_resistance(ls, ds)
    for b in range(nb):
        hp = half_soma if bp[b] < 0 else 0.5 * r[:, bp[b]]
        rax[:, 1 + b * n] = hp + 0.5 * r[:, b]
    return parent, area, rax


# ----------------------------------------------------------------------------------------------
# model dict helpers
# ----------------------------------------------------------------------------------------------
_F64 = ("cv_area", "cv_cm", "cv_raxial", "cv_vinit", "hh_gnabar", "hh_gkbar", "hh_gl", "pas_g",
        "pas_e", "syn_tau", "syn_e", "clamp_t0", "clamp_t1", "clamp_amp", "conn_delay",
        "conn_weight", "ext_time", "ext_weight")
_I64 = ("cv_off", "syn_off", "clamp_cell", "conn_src", "conn_dst", "ext_cell")
_I32 = ("cv_parent", "syn_cv", "clamp_cv", "det_cv", "conn_syn", "ext_syn")
_LIF = ("lif_tau_m", "lif_v_th", "lif_c_m", "lif_e_l", "lif_e_r", "lif_t_ref")


def finalize(m):
    """Fill defaults and coerce dtypes / contiguity.  Pure bookkeeping."""
    n_cells = int(m["n_cells"])
    m.setdefault("cv_vinit", None)
    m.setdefault("det_cv", None)
    m.setdefault("hh_ena", ENA), m.setdefault("hh_ek", EK), m.setdefault("hh_el", EL)
    m.setdefault("threshold", THRESHOLD)
    m.setdefault("dt", DT)
    for k in ("hh_gnabar", "hh_gkbar", "hh_gl", "pas_g", "pas_e"):
        m.setdefault(k, None)
    if m.get("syn_off") is None:
        m["syn_off"] = np.zeros(n_cells + 1, np.int64)
    for k, dt in (("syn_cv", np.int32), ("syn_tau", float), ("syn_e", float),
                  ("clamp_cell", np.int64), ("clamp_cv", np.int32), ("clamp_t0", float),
                  ("clamp_t1", float), ("clamp_amp", float), ("conn_src", np.int64),
                  ("conn_dst", np.int64), ("conn_syn", np.int32), ("conn_delay", float),
                  ("conn_weight", float), ("ext_cell", np.int64), ("ext_syn", np.int32),
                  ("ext_time", float), ("ext_weight", float)):
        if m.get(k) is None:
            m[k] = np.zeros(0, dt)
    for k in _F64:
        if m[k] is not None:
            m[k] = np.ascontiguousarray(m[k], dtype=np.float64)
    for k in _I64:
        m[k] = np.ascontiguousarray(m[k], dtype=np.int64)
    for k in _I32:
        if m[k] is not None:
            m[k] = np.ascontiguousarray(m[k], dtype=np.int32)
    # cell kinds: None = every cell is a multi-compartment cell
    if m.get("cell_kind") is None:
        m["cell_kind"] = None
        for k in _LIF + ("src_off", "src_time"):
            m[k] = None
    else:
        m["cell_kind"] = np.ascontiguousarray(m["cell_kind"], dtype=np.int32)
        for k in _LIF:
            m[k] = np.ascontiguousarray(m[k] if m.get(k) is not None else np.ones(n_cells), dtype=np.float64)
        m["src_off"] = np.ascontiguousarray(m["src_off"] if m.get("src_off") is not None else np.zeros(n_cells + 1), dtype=np.int64)
        m["src_time"] = np.ascontiguousarray(m["src_time"] if m.get("src_time") is not None else np.zeros(0), dtype=np.float64)
    m["n_cv"] = int(m["cv_off"][-1])
    m["n_syn"] = int(m["syn_off"][-1])
    m["n_clamp"] = len(m["clamp_cell"])
    m["n_conn"] = len(m["conn_src"])
    m["n_ext"] = len(m["ext_cell"])
    return m


def _poisson_events(rng, rate_hz, t_end_ms, syn_lo, syn_hi):
    """Homogeneous Poisson process of total rate `rate_hz` on [0, t_end), synapse uniform."""
    k = int(rng.poisson(rate_hz * t_end_ms * 1e-3))
    t = np.sort(rng.uniform(0.0, t_end_ms, k))
    s = rng.integers(syn_lo, syn_hi, k).astype(np.int32)
    return t, s


def _binary_tree(nb):
    return np.array([-1] + [(b - 1) // 2 for b in range(1, nb)], np.int64)


def _homogeneous(cfg, n_cells, nb, n, n_syn, t_end, first_cell=0):
    """Cells of configs 1-3: full binary tree of nb branches with n CVs each, HH soma, passive dendrites.
    `first_cell` shifts the per-cell seeds: cell c draws from stream [seed, first_cell + c]."""
    seed = BASE_SEED + cfg
    ncv = 1 + nb * n
    L = np.empty((n_cells, nb))
    D = np.empty((n_cells, nb))
    syn_cv = np.empty((n_cells, n_syn), np.int32)
    rngs = []
    for c in range(n_cells):
        rng = np.random.default_rng([seed, first_cell + c])
        L[c] = rng.uniform(100.0, 300.0, nb)
        D[c] = rng.uniform(0.5, 2.0, nb)
        syn_cv[c] = rng.integers(0, ncv, n_syn)
        rngs.append(rng)
    parent, area, rax = _uniform_topology_cvs(_binary_tree(nb), n, L, D)
    n_cv = n_cells * ncv
    soma = np.arange(n_cells, dtype=np.int64) * ncv
    m = dict(n_cells=n_cells,
             cv_off=np.arange(n_cells + 1, dtype=np.int64) * ncv,
             cv_parent=np.tile(parent, n_cells),
             cv_area=area.reshape(-1), cv_cm=np.full(n_cv, CM), cv_raxial=rax.reshape(-1))
    for k, v in (("hh_gnabar", GNABAR), ("hh_gkbar", GKBAR), ("hh_gl", GL)):
        a = np.zeros(n_cv)
        a[soma] = v
        m[k] = a
    g = np.full(n_cv, G_PAS)
    g[soma] = 0.0
    m["pas_g"], m["pas_e"] = g, np.full(n_cv, E_PAS)
    m["syn_off"] = np.arange(n_cells + 1, dtype=np.int64) * n_syn
    m["syn_cv"] = syn_cv.reshape(-1)
    m["syn_tau"] = np.full(n_cells * n_syn, SYN_TAU)
    m["syn_e"] = np.full(n_cells * n_syn, SYN_E)
    m["t_end"] = t_end
    return m, rngs


def _random_network(m, rngs, n_in, weight, ext_rate_hz, ext_syn_lo, ext_syn_hi, ext_weight, t_end, first_cell=0, n_global=None):
    """n_in incoming connections per cell (sources uniform, no self connection),
    connection j of a cell lands on its synapse j; delay U(5,10) ms; Poisson external events.
    n_global: the cells of `m` are cells first_cell ... of a network of n_global cells (a shard, sharded.py):
    sources are drawn over the whole network and stay global ids, exactly as when the network is generated whole."""
    n_cells = m["n_cells"]
    n_net = n_cells if n_global is None else int(n_global)
    src = np.empty((n_cells, n_in), np.int64)
    dly = np.empty((n_cells, n_in))
    et, es, ec = [], [], []
    for c, rng in enumerate(rngs):
        if n_net > 1:
            s = rng.integers(0, n_net - 1, n_in)
            src[c] = s + (s >= c + (first_cell if n_global is not None else 0))
        else:
            src[c] = 0
        dly[c] = rng.uniform(5.0, 10.0, n_in)
        if ext_rate_hz > 0:
            t, s = _poisson_events(rng, ext_rate_hz, t_end, ext_syn_lo, ext_syn_hi)
            et.append(t), es.append(s), ec.append(np.full(len(t), c, np.int64))
    if n_net > 1:
        m["conn_src"] = src.reshape(-1)
        m["conn_dst"] = np.repeat(np.arange(n_cells, dtype=np.int64), n_in)
        m["conn_syn"] = np.tile(np.arange(n_in, dtype=np.int32), n_cells)
        m["conn_delay"] = dly.reshape(-1)
        m["conn_weight"] = np.full(n_cells * n_in, weight)
    if et:
        m["ext_cell"] = np.concatenate(ec)
        m["ext_syn"] = np.concatenate(es)
        m["ext_time"] = np.concatenate(et)
        m["ext_weight"] = np.full(len(m["ext_time"]), ext_weight)
    return m


# ----------------------------------------------------------------------------------------------
# the five BASELINE.json configs
# ----------------------------------------------------------------------------------------------
def config0():
    """configs[0]: HH soma + 10-CV passive dendrite, 0.1 nA clamp 10-60 ms, 100 ms."""
    parent, area, rax, _ = cell_cvs([-1], [10], [200.0], [1.0])
    n = len(parent)
    z = np.zeros(n)
    hh = lambda v: np.concatenate([[v], z[1:]])
    g = np.full(n, G_PAS)
    g[0] = 0.0
    m = dict(n_cells=1, cv_off=[0, n], cv_parent=parent, cv_area=area, cv_cm=np.full(n, CM),
             cv_raxial=rax, hh_gnabar=hh(GNABAR), hh_gkbar=hh(GKBAR), hh_gl=hh(GL),
             pas_g=g, pas_e=np.full(n, E_PAS),
             clamp_cell=[0], clamp_cv=[0], clamp_t0=[10.0], clamp_t1=[60.0], clamp_amp=[0.1],
             t_end=100.0, name="C0 single cell")
    return finalize(m)


def config1(n_cells=1000, t_end=200.0, weight=0.01, kick_weight=0.1, ring_syn_on_soma=True):
    """configs[1]: ring of depth-4 binary-tree cells (15 branches x 20 CVs), 10 expsyn, delay 5 ms.

    Reading: the ring connection and the kick land on synapse 0, and synapse 0 sits on
    the soma; the other nine synapses are on random CVs.  With synapse 0 on a random dendritic CV
    the ring dies after one or two cells at the stated weight (0.01 uS)."""
    m, _ = _homogeneous(1, n_cells, 15, 20, 10, t_end)
    if ring_syn_on_soma:
        m["syn_cv"][::10] = 0
    i = np.arange(n_cells, dtype=np.int64)
    if n_cells > 1:
        m["conn_src"], m["conn_dst"] = i, (i + 1) % n_cells
        m["conn_syn"] = np.zeros(n_cells, np.int32)
        m["conn_delay"] = np.full(n_cells, 5.0)
        m["conn_weight"] = np.full(n_cells, weight)
    m["ext_cell"], m["ext_syn"], m["ext_time"], m["ext_weight"] = [0], [0], [1.0], [kick_weight]
    m["name"] = "C1 ring %d" % n_cells
    return finalize(m)


def config2(n_cells=10000, t_end=1000.0):
    """configs[2]: random network, 100 incoming connections + 20 Poisson (10 Hz) input synapses."""
    m, rngs = _homogeneous(2, n_cells, 15, 20, 120, t_end)
    _random_network(m, rngs, 100, 0.001, 20 * 10.0, 100, 120, 0.001, t_end)
    m["name"] = "C2 random %d" % n_cells
    return finalize(m)


def config3(n_cells=100000, t_end=200.0, driven=True, first_cell=0, n_global=None):
    """configs[3]: depth-6 trees (63 branches x 8 CVs), 50 expsyn, 50 incoming connections.
    BASELINE.json names no drive; `driven` adds 200 Hz/cell Poisson input.
    `first_cell` selects another closed network of the same population (bench.py: one per rank); with
    `n_global` the cells are instead cells first_cell ... first_cell + n_cells of ONE network of n_global cells
    (a rank's shard, generated without the rest: conn_src are global ids, shard_* fields are set)."""
    m, rngs = _homogeneous(3, n_cells, 63, 8, 50, t_end, first_cell)
    _random_network(m, rngs, 50, 0.002, 200.0 if driven else 0.0, 0, 50, 0.002, t_end, first_cell, n_global)
    m["name"] = "C3 large %d%s" % (n_cells, "" if driven else " undriven")
    if n_global is not None:
        m["shard_gid_base"], m["shard_n_global"] = int(first_cell), int(n_global)
    return finalize(m)


def config4(n_cells=50000, t_end=200.0):
    """configs[4]: heterogeneous trees: depth U{2..8}, split p=0.7, 4..40 CVs/branch, HH on soma and
    10% of dendritic CVs, passive elsewhere; 30 synapses / incoming connections."""
    seed = BASE_SEED + 4
    n_syn = 30
    parents, areas, raxs, hhs, syns, offs, rngs = [], [], [], [], [], [0], []
    for c in range(n_cells):
        rng = np.random.default_rng([seed, c])
        depth = int(rng.integers(2, 9))
        bp, lvl = [-1], [1]
        b = 0
        while b < len(bp):                      # breadth-first growth
            if lvl[b] < depth and rng.random() < 0.7:
                bp += [b, b]
                lvl += [lvl[b] + 1, lvl[b] + 1]
            b += 1
        nb = len(bp)
        ncvb = rng.integers(4, 41, nb)
        L = rng.uniform(100.0, 300.0, nb)
        D = rng.uniform(0.5, 2.0, nb)
        parent, area, rax, _ = cell_cvs(bp, ncvb, L, D)
        n = len(parent)
        hh = rng.random(n) < 0.1
        hh[0] = True
        parents.append(parent), areas.append(area), raxs.append(rax), hhs.append(hh)
        syns.append(rng.integers(0, n, n_syn).astype(np.int32))
        offs.append(offs[-1] + n)
        rngs.append(rng)
    hh = np.concatenate(hhs)
    n_cv = offs[-1]
    m = dict(n_cells=n_cells, cv_off=offs, cv_parent=np.concatenate(parents),
             cv_area=np.concatenate(areas), cv_cm=np.full(n_cv, CM),
             cv_raxial=np.concatenate(raxs),
             hh_gnabar=np.where(hh, GNABAR, 0.0), hh_gkbar=np.where(hh, GKBAR, 0.0),
             hh_gl=np.where(hh, GL, 0.0), pas_g=np.where(hh, 0.0, G_PAS),
             pas_e=np.full(n_cv, E_PAS),
             syn_off=np.arange(n_cells + 1, dtype=np.int64) * n_syn,
             syn_cv=np.concatenate(syns), syn_tau=np.full(n_cells * n_syn, SYN_TAU),
             syn_e=np.full(n_cells * n_syn, SYN_E), t_end=t_end,
             name="C4 heterogeneous %d" % n_cells)
    _random_network(m, rngs, 30, 0.002, 200.0, 0, 30, 0.002, t_end)
    return finalize(m)


def paper_ring(n_cells=1024, n_syn=10000, t_end=200.0, weight=0.05, kick_weight=0.1):
    """The paper's own single-node benchmark cell: random
    morphologies of ~130 control volumes (here: a binary tree of 7 branches with U{12..24} CVs each),
    HH soma, passive dendrites, `n_syn` exponential synapses per cell at random control volumes of
    which ONE is wired: cell i -> cell i+1 (synapse 0, delay 5 ms); cell 0 is kicked at t = 1 ms.
    Synapse-dominated: ~10,000 synapse instances against ~130 control volumes per cell."""
    seed = BASE_SEED + 5
    bp = _binary_tree(7)
    parents, areas, raxs, syns, offs = [], [], [], [], [0]
    for c in range(n_cells):
        rng = np.random.default_rng([seed, c])
        ncvb = rng.integers(12, 25, 7)
        L = rng.uniform(100.0, 300.0, 7)
        D = rng.uniform(0.5, 2.0, 7)
        parent, area, rax, _ = cell_cvs(bp, ncvb, L, D)
        n = len(parent)
        s = rng.integers(0, n, n_syn).astype(np.int32)
        s[0] = 0                                            # the wired synapse sits on the soma
        parents.append(parent), areas.append(area), raxs.append(rax), syns.append(s)
        offs.append(offs[-1] + n)
    n_cv = offs[-1]
    soma = np.asarray(offs[:-1], np.int64)
    hh = np.zeros(n_cv)
    hh[soma] = 1.0
    m = dict(n_cells=n_cells, cv_off=offs, cv_parent=np.concatenate(parents), cv_area=np.concatenate(areas),
             cv_cm=np.full(n_cv, CM), cv_raxial=np.concatenate(raxs),
             hh_gnabar=hh * GNABAR, hh_gkbar=hh * GKBAR, hh_gl=hh * GL,
             pas_g=np.where(hh > 0, 0.0, G_PAS), pas_e=np.full(n_cv, E_PAS),
             syn_off=np.arange(n_cells + 1, dtype=np.int64) * n_syn, syn_cv=np.concatenate(syns),
             syn_tau=np.full(n_cells * n_syn, SYN_TAU), syn_e=np.full(n_cells * n_syn, SYN_E),
             conn_src=np.arange(n_cells), conn_dst=(np.arange(n_cells) + 1) % n_cells,
             conn_syn=np.zeros(n_cells, np.int32), conn_delay=np.full(n_cells, 5.0),
             conn_weight=np.full(n_cells, weight),
             ext_cell=[0], ext_syn=[0], ext_time=[1.0], ext_weight=[kick_weight],
             t_end=t_end, name="paper ring %d x %d synapses" % (n_cells, n_syn))
    return finalize(m)


def config(k, **kw):
    return (config0, config1, config2, config3, config4)[k](**kw)


# ----------------------------------------------------------------------------------------------
# other cell kinds: LIF cells and spike sources beside cable cells
# ----------------------------------------------------------------------------------------------
LIF_DEFAULTS = dict(lif_tau_m=10.0, lif_v_th=-50.0, lif_c_m=0.25, lif_e_l=-65.0, lif_e_r=-70.0, lif_t_ref=2.0)


def mixed_network(seed=0, n_cable=6, n_lif=8, n_src=4, t_end=60.0, rate_hz=60.0, n_in=4):
    """A small network of all three cell kinds: Poisson spike sources drive LIF cells and cable cells (configs[1]
    morphologies), LIF cells and cable cells project onto each other.  Cells are numbered sources, LIF, cable.
    A LIF / source cell owns one (unused) control volume; a LIF cell's events target its synapse range (n_in
    targets), an event's weight is a charge [pC] for LIF cells and a conductance [uS] for cable cells."""
    rng = np.random.default_rng([BASE_SEED, 99, seed])
    cab, _ = _homogeneous(1, n_cable, 15, 20, n_in, t_end)
    n_cells = n_src + n_lif + n_cable
    n_other = n_src + n_lif
    ncv_c = int(cab["cv_off"][1])
    off = np.concatenate([np.arange(n_other + 1), n_other + cab["cv_off"][1:]])
    one = lambda v, arr: np.concatenate([np.full(n_other, v), arr])
    m = dict(n_cells=n_cells, cv_off=off, cv_parent=np.concatenate([np.full(n_other, -1, np.int32), cab["cv_parent"]]),
             cv_area=one(100.0, cab["cv_area"]), cv_cm=one(1.0, cab["cv_cm"]), cv_raxial=one(1.0, cab["cv_raxial"]),
             cv_vinit=one(-65.0, np.full(n_cable * ncv_c, -65.0)),
             hh_gnabar=one(0.0, cab["hh_gnabar"]), hh_gkbar=one(0.0, cab["hh_gkbar"]), hh_gl=one(0.0, cab["hh_gl"]),
             pas_g=one(0.0, cab["pas_g"]), pas_e=one(-65.0, cab["pas_e"]),
             syn_off=np.concatenate([np.zeros(n_src + 1, np.int64), np.arange(1, n_lif + n_cable + 1) * n_in]),
             syn_cv=np.concatenate([np.zeros(n_lif * n_in, np.int32), np.zeros(n_cable * n_in, np.int32)]),
             syn_tau=np.full((n_lif + n_cable) * n_in, SYN_TAU), syn_e=np.full((n_lif + n_cable) * n_in, SYN_E),
             cell_kind=np.concatenate([np.full(n_src, 2), np.full(n_lif, 1), np.zeros(n_cable)]).astype(np.int32),
             t_end=t_end, name="mixed network %d+%d+%d" % (n_src, n_lif, n_cable))
    for k, v in LIF_DEFAULTS.items():
        m[k] = np.full(n_cells, v) * (1.0 if k != "lif_tau_m" else 1.0) + (rng.uniform(-0.5, 0.5, n_cells) if k == "lif_tau_m" else 0.0)
    # Poisson schedules of the sources
    times, soff = [], [0]
    for c in range(n_cells):
        if c < n_src:
            k = int(rng.poisson(rate_hz * t_end * 1e-3))
            times.append(np.sort(rng.uniform(0.0, t_end, k)))
        else:
            times.append(np.zeros(0))
        soff.append(soff[-1] + len(times[-1]))
    m["src_off"], m["src_time"] = np.array(soff), np.concatenate(times)
    # connections: target synapse j of every LIF / cable cell gets one source: sources and LIF cells drive everybody
    src, dst, syn, dly, w = [], [], [], [], []
    for c in range(n_src, n_cells):
        for j in range(n_in):
            s = int(rng.integers(0, n_other))
            if s == c:
                s = (s + 1) % n_other
            src.append(s), dst.append(c), syn.append(j), dly.append(float(rng.uniform(1.0, 4.0)))
            w.append(float(rng.uniform(1.5, 3.0)) if c < n_other else float(rng.uniform(0.005, 0.02)))
    # cable cells project back onto the LIF cells
    for c in range(n_other, n_cells):
        for j in range(2):
            src.append(c), dst.append(int(rng.integers(n_src, n_other))), syn.append(int(rng.integers(0, n_in)))
            dly.append(float(rng.uniform(1.0, 4.0))), w.append(float(rng.uniform(2.0, 4.0)))
    m.update(conn_src=src, conn_dst=dst, conn_syn=syn, conn_delay=dly, conn_weight=w)
    return finalize(m)


# ----------------------------------------------------------------------------------------------
# small arbitrary models for parity / pin tests
# ----------------------------------------------------------------------------------------------
def random_parent(rng, n, kind="random"):
    """A valid parent array (parent < index, root -1) of a given shape family."""
    p = np.full(n, -1, np.int32)
    for i in range(1, n):
        if kind == "chain":
            p[i] = i - 1
        elif kind == "star":
            p[i] = 0
        elif kind == "binary":
            p[i] = (i - 1) // 2
        elif kind == "bushy":                     # many short branches
            p[i] = rng.integers(max(0, i - 3), i)
        else:
            p[i] = rng.integers(0, i)
    return p


def random_model(seed, n_cells=5, max_cv=40, kinds=("random", "chain", "star", "binary", "bushy"),
                 p_hh=0.3, p_pas=0.8, max_syn=6, n_conn=None, n_ext=None, n_clamp=None,
                 t_end=20.0, dt=DT, strong=True, per_syn_params=True, vinit=True, det_random=True):
    """A small network with arbitrary trees and every feature of arb_desc switched on."""
    rng = np.random.default_rng([BASE_SEED, 77, seed])
    offs, parents = [0], []
    for c in range(n_cells):
        n = int(rng.integers(1, max_cv + 1))
        parents.append(random_parent(rng, n, kinds[int(rng.integers(len(kinds)))]))
        offs.append(offs[-1] + n)
    n_cv = offs[-1]
    off = np.array(offs)
    area = rng.uniform(50.0, 600.0, n_cv)
    hh = rng.random(n_cv) < p_hh
    hh[off[:-1]] |= rng.random(n_cells) < 0.8
    pas = (~hh) & (rng.random(n_cv) < p_pas)
    nsyn = rng.integers(0, max_syn + 1, n_cells)
    if n_cells > 1 and max_syn > 0:
        nsyn = np.maximum(nsyn, 1)
    syn_off = np.concatenate([[0], np.cumsum(nsyn)])
    syn_cv = np.concatenate([rng.integers(0, off[c + 1] - off[c], nsyn[c]) for c in range(n_cells)]
                            + [np.zeros(0, np.int64)])
    ns = int(syn_off[-1])
    m = dict(n_cells=n_cells, cv_off=off, cv_parent=np.concatenate(parents), cv_area=area,
             cv_cm=rng.uniform(0.9, 2.0, n_cv), cv_raxial=rng.uniform(0.5, 40.0, n_cv),
             cv_vinit=rng.uniform(-70.0, -55.0, n_cv) if vinit else None,
             hh_gnabar=np.where(hh, rng.uniform(0.08, 0.14, n_cv), 0.0),
             hh_gkbar=np.where(hh, rng.uniform(0.03, 0.04, n_cv), 0.0),
             hh_gl=np.where(hh, rng.uniform(2e-4, 4e-4, n_cv), 0.0),
             pas_g=np.where(pas, rng.uniform(5e-6, 5e-4, n_cv), 0.0),
             pas_e=rng.uniform(-70.0, -60.0, n_cv),
             syn_off=syn_off, syn_cv=syn_cv,
             syn_tau=rng.uniform(0.5, 5.0, ns) if per_syn_params else np.full(ns, SYN_TAU),
             syn_e=rng.uniform(-10.0, 10.0, ns) if per_syn_params else np.full(ns, SYN_E),
             t_end=t_end, dt=dt, threshold=float(rng.uniform(-20.0, 0.0)),
             name="random model %d" % seed)
    if det_random:
        m["det_cv"] = np.array([rng.integers(0, off[c + 1] - off[c]) for c in range(n_cells)])
    w = 0.004 if strong else 0.001   # explicit currents (R1) need dt*g/C < 2
    has_syn = np.flatnonzero(nsyn > 0)
    if n_conn is None:
        n_conn = 3 * n_cells
    if len(has_syn) and n_conn:
        dst = has_syn[rng.integers(0, len(has_syn), n_conn)]
        m["conn_src"] = rng.integers(0, n_cells, n_conn)
        m["conn_dst"] = dst
        m["conn_syn"] = np.array([rng.integers(0, nsyn[d]) for d in dst])
        m["conn_delay"] = rng.uniform(0.5, 4.0, n_conn)
        m["conn_weight"] = rng.uniform(0.2 * w, w, n_conn)
    if n_ext is None:
        n_ext = 6 * n_cells
    if len(has_syn) and n_ext:
        ec = has_syn[rng.integers(0, len(has_syn), n_ext)]
        es = np.array([rng.integers(0, nsyn[d]) for d in ec])
        t = rng.uniform(0.0, t_end, n_ext)
        k = n_ext // 4                            # a quarter land exactly on grid points
        t[:k] = np.round(t[:k] / dt) * dt
        if n_ext >= 8:                            # simultaneous events: same synapse / same cell
            ec[k], es[k], t[k] = ec[k + 1], es[k + 1], t[k + 1]
            ec[k + 2], t[k + 2] = ec[k + 3], t[k + 3]
            es[k + 2] = rng.integers(0, nsyn[ec[k + 3]])
        m["ext_cell"], m["ext_syn"], m["ext_time"] = ec, es, t
        m["ext_weight"] = rng.uniform(0.2 * w, 2 * w, n_ext)
    if n_clamp is None:
        n_clamp = max(1, n_cells // 2)
    if n_clamp:
        cc = rng.integers(0, n_cells, n_clamp)
        m["clamp_cell"] = cc
        m["clamp_cv"] = np.array([rng.integers(0, off[c + 1] - off[c]) for c in cc])
        t0 = rng.uniform(0.0, 0.6 * t_end, n_clamp)
        m["clamp_t0"] = t0
        m["clamp_t1"] = t0 + rng.uniform(0.1 * t_end, 0.5 * t_end, n_clamp)
        m["clamp_amp"] = rng.uniform(-0.05, 0.4, n_clamp)
    return finalize(m)


def passive_cable(n, g_pas=1e-4, area=100.0, rax=5.0, cm=1.0, e_pas=-65.0, i_inj=0.0, t_end=250.0,
                  dt=DT, vinit=None):
    """Unbranched chain of n identical passive CVs, sealed ends, optional constant current into CV 0."""
    m = dict(n_cells=1, cv_off=[0, n], cv_parent=np.arange(-1, n - 1), cv_area=np.full(n, area),
             cv_cm=np.full(n, cm), cv_raxial=np.full(n, rax), pas_g=np.full(n, g_pas),
             pas_e=np.full(n, e_pas), cv_vinit=vinit, t_end=t_end, dt=dt, name="passive cable")
    if i_inj != 0.0:
        m.update(clamp_cell=[0], clamp_cv=[0], clamp_t0=[0.0], clamp_t1=[1e300],
                 clamp_amp=[i_inj])
    return finalize(m)


def take_cells(m, cells):
    """Sub-model made of the given cells only, WITHOUT connections (keeps their external events
    and clamps).  Valid as an independent reference only while no network event has arrived."""
    cells = np.asarray(cells, np.int64)
    off = m["cv_off"]
    idx = np.concatenate([np.arange(off[c], off[c + 1]) for c in cells])
    out = dict(n_cells=len(cells),
               cv_off=np.concatenate([[0], np.cumsum(off[cells + 1] - off[cells])]),
               t_end=m["t_end"], dt=m["dt"], threshold=m["threshold"],
               hh_ena=m["hh_ena"], hh_ek=m["hh_ek"], hh_el=m["hh_el"],
               name=m.get("name", "") + " [cells]")
    for k in ("cv_parent", "cv_area", "cv_cm", "cv_raxial", "cv_vinit", "hh_gnabar", "hh_gkbar",
              "hh_gl", "pas_g", "pas_e"):
        out[k] = None if m[k] is None else m[k][idx]
    so = m["syn_off"]
    sidx = np.concatenate([np.arange(so[c], so[c + 1]) for c in cells] + [np.zeros(0, np.int64)])
    out["syn_off"] = np.concatenate([[0], np.cumsum(so[cells + 1] - so[cells])])
    for k in ("syn_cv", "syn_tau", "syn_e"):
        out[k] = m[k][sidx]
    if m["det_cv"] is not None:
        out["det_cv"] = m["det_cv"][cells]
    remap = {int(c): i for i, c in enumerate(cells)}
    for cellkey, keys in (("ext_cell", ("ext_syn", "ext_time", "ext_weight")),
                          ("clamp_cell", ("clamp_cv", "clamp_t0", "clamp_t1", "clamp_amp"))):
        sel = np.flatnonzero(np.isin(m[cellkey], cells))
        out[cellkey] = np.array([remap[int(c)] for c in m[cellkey][sel]], np.int64)
        for k in keys:
            out[k] = m[k][sel]
    return finalize(out)
