"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element, on the
same seeded inputs.  Tolerances are BASELINE.json north_star's:
  * V and gate states after each single step: |d| <= 1e-12 * max(|ref|, 1)   (reading R17)
  * passive runs after 10,000 steps: max |dV| <= 1e-9 mV
  * active networks: identical spike counts per cell, spike times within 1e-3 ms.
"Each single step" is checked from a common state: the oracle's state is loaded into the GPU model
before every step (arb_set_state), so the bound is on one step of arithmetic, not on accumulated
divergence of a nonlinear system.  Free-running trajectories are checked as well, with the
tolerance DESIGN.md derives for them.
"""
import numpy as np
import pytest

from paper_1901_07454_b200 import workloads as W

pytestmark = pytest.mark.gpu

DT = 0.025
STEP_TOL = 1e-12


@pytest.fixture(scope="module")
def B():
    import torch
    assert torch.cuda.is_available(), "these tests need a CUDA device"
    from paper_1901_07454_b200 import binding
    binding.lib()
    return binding


@pytest.fixture(params=["default", "groups", "units"], autouse=True)
def layout(request, B):
    """Every test runs under three layouts: the default (cells of a topology class of >= 4 cells in
    cell-interleaved groups, the rest in branch-interleaved units), every cell in groups, no groups."""
    B.LAYOUT_DEFAULTS["layout_group_min_cells"] = {"default": 0, "groups": 1, "units": 2 ** 31}[request.param]
    yield request.param
    B.LAYOUT_DEFAULTS.clear()


def rel(a, b):
    return float(np.max(np.abs(a - b) / np.maximum(np.abs(b), 1.0))) if len(a) else 0.0


def rel_pure(a, b):
    nz = b != 0
    assert np.all(a[~nz] == 0)
    return float(np.max(np.abs(a[nz] - b[nz]) / np.abs(b[nz]))) if nz.any() else 0.0


def state_of(x):
    return (x.voltage(),) + tuple(x.gates()) + (x.syn_g(),)


def check_state(g, o, tol, what=""):
    gs, os_ = state_of(g), state_of(o)
    for name, a, b in zip(("V", "m", "h", "n"), gs, os_):
        assert rel(a, b) <= tol, "%s %s: %g" % (what, name, rel(a, b))
    assert rel_pure(gs[4], os_[4]) <= tol, "%s g: %g" % (what, rel_pure(gs[4], os_[4]))


def check_spikes(g, o, n_cells, tol=1e-3):
    gc, gt = g.spikes()
    oc, ot = o.spikes()
    assert np.array_equal(np.bincount(gc, minlength=n_cells), np.bincount(oc, minlength=n_cells))
    # per cell, in time order
    gi, oi = np.lexsort((gt, gc)), np.lexsort((ot, oc))
    assert np.array_equal(gc[gi], oc[oi])
    if len(gt):
        assert np.max(np.abs(gt[gi] - ot[oi])) <= tol
    return len(gc)


def lockstep(B, orc, m, nsteps, fused=0, resync=True, tol=STEP_TOL, linearised=False):
    """Advance both one grid step at a time and compare after every step."""
    g, o = B.Model(m), orc.Oracle(m)
    if fused:
        g.set_option(B.ARB_OPT_FUSED_STEPS, fused)
    if linearised:
        g.set_option(B.ARB_OPT_LINEARISED, 1)
        o.set_linearised(True)
    check_state(g, o, 1e-15, "initial")
    dt = m["dt"]
    for k in range(1, nsteps + 1):
        g.advance(k * dt, dt)
        o.advance(k * dt, dt)
        check_state(g, o, tol, "step %d" % k)
        if resync:
            v, (hm, hh, hn), sg = o.voltage(), o.gates(), o.syn_g()
            g.set_state(v, hm, hh, hn, sg)
            o.set_state(v, hm, hh, hn, sg)
    n = check_spikes(g, o, m["n_cells"])
    assert tuple(g.probe(B.ARB_PROBE_NSTEPS)) == tuple(o.probe(orc.PROBE_NSTEPS))
    g.close()
    return n


# ---------------------------------------------------------------------------------------------
# per-step parity
# ---------------------------------------------------------------------------------------------
def test_config0_every_step(B, orc):
    """configs[0], first 2,000 steps (clamp on at 10 ms -> spikes inside the window)."""
    assert lockstep(B, orc, W.config0(), 2000) >= 2


def test_config0_free_running_2000_steps(B, orc):
    """Same without re-synchronising: accumulated divergence stays tiny on a single cell."""
    lockstep(B, orc, W.config0(), 2000, resync=False, tol=1e-10)


def test_config1_cut_every_step(B, orc):
    """64-cell cut of configs[1], first 2,000 steps, ring spikes travelling through it."""
    assert lockstep(B, orc, W.config1(n_cells=64, t_end=50.0), 2000) >= 5


@pytest.mark.parametrize("seed", range(1, 9))
def test_random_models_every_step(B, orc, seed):
    """Arbitrary trees (chains, stars, bushy, binary, random), every mechanism, events on and off the
    grid, simultaneous events, clamps, random detectors: 400 steps in lockstep."""
    lockstep(B, orc, W.random_model(seed, n_cells=7, t_end=10.0), 400)


@pytest.mark.parametrize("fused", [1, 7])
def test_launch_granularity_does_not_change_results(B, orc, fused):
    m = W.random_model(3, n_cells=9, t_end=12.0)
    res = []
    for f in (0, fused):
        g = B.Model(m)
        if f:
            g.set_option(B.ARB_OPT_FUSED_STEPS, f)
        g.advance(12.0, DT)
        res.append(state_of(g) + g.spikes())
        g.close()
    for a, b in zip(*res):
        assert np.array_equal(a, b)


# ---------------------------------------------------------------------------------------------
# the conductance-linearised step (ARB_OPT_LINEARISED): per-step parity at 1e-12
# ---------------------------------------------------------------------------------------------
def test_linearised_config0_every_step(B, orc):
    assert lockstep(B, orc, W.config0(), 2000, linearised=True) >= 2


def test_linearised_config1_cut_every_step(B, orc):
    assert lockstep(B, orc, W.config1(n_cells=32, t_end=30.0), 1000, linearised=True) >= 2


@pytest.mark.parametrize("seed", range(1, 7))
def test_linearised_random_models_every_step(B, orc, seed):
    """Arbitrary trees, every mechanism, per-synapse tau and e, events on and off the grid (event-split sub-steps
    re-assemble with the cell's own C/delta), clamps."""
    lockstep(B, orc, W.random_model(seed, n_cells=7, t_end=10.0), 400, linearised=True)


def test_linearised_heterogeneous_cut_every_step(B, orc):
    lockstep(B, orc, W.config4(n_cells=30, t_end=10.0), 200, linearised=True)


def test_linearised_network_spikes_and_switching(B, orc):
    """A spiking network cut, free running: identical spike counts, times within 1e-3 ms; the option can be
    switched between calls (coefficients are rebuilt) and is stable at a step where the explicit one diverges."""
    m = W.config3(n_cells=96, t_end=40.0)
    m["conn_weight"] = m["conn_weight"] * 4
    m["ext_weight"] = m["ext_weight"] * 4
    g, o = B.Model(m), orc.Oracle(m, threads=4)
    g.set_option(B.ARB_OPT_LINEARISED, 1)
    o.set_linearised(True)
    g.advance(20.0, DT), o.advance(20.0, DT)
    g.set_option(B.ARB_OPT_LINEARISED, 0)
    o.set_linearised(False)
    g.advance(30.0, DT), o.advance(30.0, DT)
    g.set_option(B.ARB_OPT_LINEARISED, 1)
    o.set_linearised(True)
    g.advance(40.0, DT), o.advance(40.0, DT)
    assert check_spikes(g, o, 96) > 20
    assert rel(g.voltage(), o.voltage()) < 1e-6
    g.close()
    g = B.Model(W.config0())
    g.set_option(B.ARB_OPT_LINEARISED, 1)
    g.advance(100.0, 1.0)                       # dt = 1 ms: test_divergence_is_reported shows the explicit step blowing up
    assert np.all(np.abs(g.voltage()) < 200.0)
    g.close()


# ---------------------------------------------------------------------------------------------
# passive run, 10,000 steps
# ---------------------------------------------------------------------------------------------
def test_passive_10000_steps(B, orc):
    rng = np.random.default_rng(3)
    m = W.config1(n_cells=24, t_end=250.0)
    for k in ("hh_gnabar", "hh_gkbar", "hh_gl"):
        m[k] = None                                         # passive everywhere
    m["pas_g"] = np.full(m["n_cv"], W.G_PAS)
    m["cv_vinit"] = rng.uniform(-80.0, -50.0, m["n_cv"])
    m.update(clamp_cell=[0, 5], clamp_cv=[0, 17], clamp_t0=[20.0, 0.0], clamp_t1=[120.0, 1e9], clamp_amp=[0.05, -0.02])
    m = W.finalize(m)
    g, o = B.Model(m), orc.Oracle(m)
    g.advance(250.0, DT)
    o.advance(250.0, DT)
    assert g.probe(B.ARB_PROBE_NSTEPS)[0] == 10000
    assert np.max(np.abs(g.voltage() - o.voltage())) <= 1e-9
    g.close()


# ---------------------------------------------------------------------------------------------
# active networks: spike counts per cell and spike times
# ---------------------------------------------------------------------------------------------
def run_both(B, orc, m, t_end, threads=4):
    g, o = B.Model(m), orc.Oracle(m, threads=threads)
    g.advance(t_end, m["dt"])
    o.advance(t_end, m["dt"])
    return g, o


def test_ring_network_spikes(B, orc):
    m = W.config1(n_cells=40, t_end=260.0)
    g, o = run_both(B, orc, m, 260.0)
    assert check_spikes(g, o, 40) >= 44                      # more than one lap
    g.close()


def test_random_network_cut_spikes(B, orc):
    m = W.config2(n_cells=150, t_end=120.0)
    g, o = run_both(B, orc, m, 120.0)
    check_spikes(g, o, 150)
    assert g.stats()["events_delivered"] > 1000
    assert tuple(g.probe(B.ARB_PROBE_NSTEPS)) == tuple(o.probe(orc.PROBE_NSTEPS))
    g.close()


def test_large_config_cut_spikes(B, orc):
    m = W.config3(n_cells=96, t_end=60.0)
    # the stated drive leaves a 96-cell cut silent; scale the weights so that it fires
    m["conn_weight"] = m["conn_weight"] * 4
    m["ext_weight"] = m["ext_weight"] * 4
    g, o = run_both(B, orc, m, 60.0)
    assert check_spikes(g, o, 96) > 20
    g.close()


def test_stream_mode_hot_groups_first(B, orc):
    """One launch per grid step (state through HBM every step).  Groups with an event in the coming
    step are integrated first (ARB_OPT_HOT_FIRST); the order in which groups are integrated must not
    change a bit, and the run must match the oracle."""
    m = W.config3(n_cells=200, t_end=30.0)
    m["conn_weight"] = m["conn_weight"] * 4
    m["ext_weight"] = m["ext_weight"] * 4
    o = orc.Oracle(m, threads=4)
    o.advance(30.0, m["dt"])
    res = []
    for hot in (1, 0):
        g = B.Model(m)
        g.set_option(B.ARB_OPT_FUSED_STEPS, 1)
        g.set_option(B.ARB_OPT_HOT_FIRST, hot)
        for t in (7.5, 30.0):
            g.advance(t, m["dt"])
        assert check_spikes(g, o, 200) > 20
        assert rel(g.voltage(), o.voltage()) < 1e-6
        assert tuple(g.probe(B.ARB_PROBE_NSTEPS)) == tuple(o.probe(orc.PROBE_NSTEPS))
        res.append(state_of(g) + g.spikes())
        g.close()
    for a, b in zip(*res):
        assert np.array_equal(a, b)


def test_paper_ring_cell_many_synapses(B, orc):
    """SURVEY.md 8(f) NEXT-1, first cut: the paper's ring cell (~130 CVs, 10,000 exponential synapses
    each, one of them wired).  Functional parity only: such cells run on the block-unit
    kernel; a kernel designed for the synapse-dominated case is the next step."""
    m = W.paper_ring(n_cells=6, n_syn=10000, t_end=30.0)
    # a few hundred extra events so that more than one synapse per cell carries conductance
    rng = np.random.default_rng(5)
    m["ext_cell"] = np.concatenate([m["ext_cell"], rng.integers(0, 6, 300)])
    m["ext_syn"] = np.concatenate([m["ext_syn"], rng.integers(0, 10000, 300).astype(np.int32)])
    m["ext_time"] = np.concatenate([m["ext_time"], rng.uniform(0.0, 25.0, 300)])
    m["ext_weight"] = np.concatenate([m["ext_weight"], rng.uniform(0.0005, 0.004, 300)])
    m = W.finalize(m)
    g, o = run_both(B, orc, m, 30.0)
    assert check_spikes(g, o, 6) >= 4
    assert rel(g.voltage(), o.voltage()) < 1e-6
    assert rel_pure(g.syn_g(), o.syn_g()) < 1e-9
    g.close()


def test_many_synapses_key_reduction_every_step(B, orc):
    """Cells with thousands of synapses whose tau and e differ from synapse to synapse: the block-unit
    kernel sums the currents of a control volume by a warp key reduction instead of in
    index order, so this is the per-step parity case for that path, with events on and off the grid
    (event-split sub-steps take its general variant)."""
    m = W.paper_ring(n_cells=3, n_syn=3000, t_end=10.0)
    rng = np.random.default_rng(7)
    m["syn_tau"] = rng.uniform(1.0, 4.0, m["n_syn"])
    m["syn_e"] = rng.uniform(-20.0, 10.0, m["n_syn"])
    n_ev = 2000
    m["ext_cell"] = np.concatenate([m["ext_cell"], rng.integers(0, 3, n_ev)])
    m["ext_syn"] = np.concatenate([m["ext_syn"], rng.integers(0, 3000, n_ev).astype(np.int32)])
    t_ev = rng.uniform(0.0, 5.0, n_ev)
    t_ev[::3] = np.round(t_ev[::3] / DT) * DT          # a third of them on grid points
    m["ext_time"] = np.concatenate([m["ext_time"], t_ev])
    m["ext_weight"] = np.concatenate([m["ext_weight"], rng.uniform(0.0001, 0.001, n_ev)])
    m = W.finalize(m)
    lockstep(B, orc, m, 200)


def _many_synapse_runs(n_cells, n_syn, two_kinds):
    """Ring cells whose synapses share (tau, e) per control volume: the library keeps one conductance per run."""
    m = W.paper_ring(n_cells=n_cells, n_syn=n_syn, t_end=10.0)
    rng = np.random.default_rng(11)
    if two_kinds:                                  # two kinds of synapse on every control volume: two runs per CV
        kind = rng.integers(0, 2, m["n_syn"])
        m["syn_tau"] = np.where(kind == 0, 2.0, 3.5)
        m["syn_e"] = np.where(kind == 0, 0.0, -70.0)
    n_ev = 1500
    m["ext_cell"] = np.concatenate([m["ext_cell"], rng.integers(0, n_cells, n_ev)])
    m["ext_syn"] = np.concatenate([m["ext_syn"], rng.integers(0, n_syn, n_ev).astype(np.int32)])
    t_ev = rng.uniform(0.0, 5.0, n_ev)
    t_ev[::3] = np.round(t_ev[::3] / DT) * DT          # a third of them on grid points
    m["ext_time"] = np.concatenate([m["ext_time"], t_ev])
    m["ext_weight"] = np.concatenate([m["ext_weight"], rng.uniform(0.0001, 0.001, n_ev)])
    return W.finalize(m)


@pytest.mark.parametrize("two_kinds", [False, True])
def test_synapse_runs_every_step(B, orc, two_kinds):
    """SURVEY.md 8(f) NEXT-1, second half (R22): cells with >= 1,024 synapses keep one conductance per run of
    synapses on one control volume with equal (tau, e); the individual g_j are lazy records.  Per-step parity of V, gates
    and EVERY synapse's g against the oracle, the state re-injected every step (arb_set_state rebuilds the run sums)."""
    lockstep(B, orc, _many_synapse_runs(3, 2500, two_kinds), 200)


def test_synapse_runs_free_running_and_round_trip(B, orc):
    """The same cells free-running for 400 steps (lazy records decay over many steps without being touched), then
    read-back -> arb_set_state -> read-back returns the same conductances."""
    m = _many_synapse_runs(4, 2000, True)
    g, o = run_both(B, orc, m, 10.0)
    assert g.stats()["block_units"] == 0           # merged, the cells fit a forest (or a group): no block units
    g0 = g.syn_g()
    assert np.count_nonzero(g0) > 500
    assert rel_pure(g0, o.syn_g()) < 1e-9
    assert rel(g.voltage(), o.voltage()) < 1e-6
    g.set_state(syn_g=g0)
    assert rel_pure(g.syn_g(), g0) < 1e-15
    g.close()


@pytest.mark.parametrize("scale", [0.1, 0.01])
def test_fine_discretisation_split_steps(B, orc, scale):
    """Control volumes 10 x / 100 x shorter than the configs' (areas and axial resistances scaled): sigma dt / C rises from
    ~50 to ~5e3 / ~5e5, where an elimination loses log10(sigma dt / C) digits to cancellation - the oracle's textbook
    recurrence as much as the kernels' re-elimination of event-split sub-steps.  Per-step parity with
    events on and off the grid, tolerance scaled with the conditioning: 1e-15 sigma dt / C (tolerance
    derivation; measured 2e-16 and 7e-17 times the ratio)."""
    m = W.config1(n_cells=8, t_end=5.0)
    m["cv_area"] = m["cv_area"] * scale
    m["cv_raxial"] = m["cv_raxial"] * scale
    rng = np.random.default_rng(3)
    n_ev = 400
    m["ext_cell"] = np.concatenate([m["ext_cell"], rng.integers(0, 8, n_ev)])
    m["ext_syn"] = np.concatenate([m["ext_syn"], rng.integers(0, 10, n_ev).astype(np.int32)])
    t_ev = rng.uniform(0.0, 2.0, n_ev)
    t_ev[::4] = np.round(t_ev[::4] / DT) * DT
    m["ext_time"] = np.concatenate([m["ext_time"], t_ev])
    m["ext_weight"] = np.concatenate([m["ext_weight"], rng.uniform(1e-5, 1e-4, n_ev) * scale])
    m = W.finalize(m)
    cap = m["cv_cm"] * m["cv_area"] * 1e-5
    ratio = float(np.max(DT / (m["cv_raxial"][1:] * cap[1:])))
    assert ratio > 1e3
    lockstep(B, orc, m, 80, tol=max(STEP_TOL, 1e-15 * ratio))


def test_heterogeneous_cut_spikes(B, orc):
    m = W.config4(n_cells=120, t_end=60.0)
    g, o = run_both(B, orc, m, 60.0)
    assert check_spikes(g, o, 120) > 20
    assert rel(g.voltage(), o.voltage()) < 1e-6
    g.close()


def test_heterogeneous_cut_every_step(B, orc):
    lockstep(B, orc, W.config4(n_cells=40, t_end=10.0), 300)


# ---------------------------------------------------------------------------------------------
# edge cases
# ---------------------------------------------------------------------------------------------
def _simple(parent, n_cells=1, **kw):
    n = len(parent)
    m = dict(n_cells=n_cells, cv_off=np.arange(n_cells + 1) * n, cv_parent=np.tile(parent, n_cells),
             cv_area=np.full(n * n_cells, 120.0), cv_cm=np.full(n * n_cells, 1.0),
             cv_raxial=np.full(n * n_cells, 4.0), pas_g=np.full(n * n_cells, 2e-4),
             pas_e=np.full(n * n_cells, -65.0), t_end=5.0)
    hh = np.zeros(n * n_cells)
    hh[::n] = 1
    m.update(hh_gnabar=hh * W.GNABAR, hh_gkbar=hh * W.GKBAR, hh_gl=hh * W.GL)
    m.update(kw)
    return W.finalize(m)


def test_single_compartment_cells(B, orc):
    m = _simple([-1], n_cells=300, clamp_cell=np.arange(0, 300, 3), clamp_cv=np.zeros(100, np.int32),
                clamp_t0=np.full(100, 0.5), clamp_t1=np.full(100, 4.0), clamp_amp=np.linspace(0.01, 0.3, 100))
    lockstep(B, orc, m, 200)


def test_long_chain_is_cut_into_pieces(B, orc):
    """3,000-CV unbranched cable: longer than one branch piece (1,024) and than a cell block."""
    n = 3000
    lockstep(B, orc, _simple(np.arange(-1, n - 1), clamp_cell=[0], clamp_cv=[n // 2], clamp_t0=[0.0], clamp_t1=[9.0], clamp_amp=[0.4]), 60)


def test_wide_star_and_deep_comb(B, orc):
    star = np.zeros(700, np.int32)
    star[0] = -1
    lockstep(B, orc, _simple(star, clamp_cell=[0], clamp_cv=[0], clamp_t0=[0.0], clamp_t1=[9.0], clamp_amp=[0.3]), 40)
    # comb: a backbone with a one-CV tooth on every node -> one level per backbone node
    nb = 150
    par = [-1]
    back = 0
    for _ in range(nb):
        par.append(back)          # tooth
        par.append(back)          # next backbone node
        back = len(par) - 1
    lockstep(B, orc, _simple(np.array(par, np.int32), clamp_cell=[0], clamp_cv=[3], clamp_t0=[0.0], clamp_t1=[9.0], clamp_amp=[0.2]), 40)


def test_two_topology_classes_with_partial_groups(B, orc):
    """Two tree shapes, 6 and 7 cells each: every class has a full cell group and a partly filled one
    (padding lanes), the cells differ in geometry, synapses sit on shared and on branch-point CVs, and
    a clamp shares the soma with the HH mechanism (the point currents meet on one control volume)."""
    rng = np.random.default_rng(77)
    par_a = np.array([-1, 0, 1, 2, 2, 4, 3, 6, 6, 5], np.int32)             # two forks
    par_b = np.array([-1, 0, 0, 0, 1, 4, 5, 2, 7, 3, 9, 10], np.int32)       # three-way fork at the soma
    cells = [par_a] * 6 + [par_b] * 7
    off = np.concatenate([[0], np.cumsum([len(p_) for p_ in cells])])
    n_cv, n_cells = int(off[-1]), len(cells)
    hh = np.zeros(n_cv)
    hh[off[:-1]] = 1
    hh[off[:-1] + 4] = 1                                                     # a second HH CV per cell
    n_syn = 6
    syn_cv = np.concatenate([np.array([0, 0, 2, 4, 4, len(p_) - 1], np.int32) for p_ in cells])
    m = dict(n_cells=n_cells, cv_off=off, cv_parent=np.concatenate(cells),
             cv_area=rng.uniform(60.0, 200.0, n_cv), cv_cm=np.full(n_cv, 1.0), cv_raxial=rng.uniform(2.0, 8.0, n_cv),
             hh_gnabar=hh * W.GNABAR, hh_gkbar=hh * W.GKBAR, hh_gl=hh * W.GL,
             pas_g=np.where(hh > 0, 0.0, 2e-4), pas_e=np.full(n_cv, -65.0),
             syn_off=np.arange(n_cells + 1) * n_syn, syn_cv=syn_cv, syn_tau=np.full(n_cells * n_syn, 2.0),
             syn_e=np.zeros(n_cells * n_syn),
             clamp_cell=[0, 7, 12], clamp_cv=[0, 0, 4], clamp_t0=[0.5, 1.0, 0.0], clamp_t1=[6.0, 7.0, 9.0],
             clamp_amp=[0.3, 0.25, 0.2],
             ext_cell=rng.integers(0, n_cells, 60), ext_syn=rng.integers(0, n_syn, 60),
             ext_time=np.round(rng.uniform(0.0, 9.0, 60), 2) + rng.choice([0.0, 0.0031], 60),
             ext_weight=rng.uniform(0.001, 0.02, 60),
             conn_src=np.arange(n_cells), conn_dst=(np.arange(n_cells) + 1) % n_cells,
             conn_syn=np.zeros(n_cells, np.int32), conn_delay=np.full(n_cells, 1.0), conn_weight=np.full(n_cells, 0.02),
             t_end=10.0)
    lockstep(B, orc, W.finalize(m), 400)


def test_two_models_alive_at_once(B, orc):
    """Two models with different shared-memory footprints, created one after the other and advanced
    alternately in both launch granularities: nothing in the library is per-process state."""
    ma = W.config3(n_cells=40, t_end=12.0)
    ma["ext_weight"] = ma["ext_weight"] * 4
    mb = W.config1(n_cells=12, t_end=12.0)
    ga, gb = B.Model(ma), B.Model(mb)
    ga.set_option(B.ARB_OPT_FUSED_STEPS, 1)
    oa, ob = orc.Oracle(ma), orc.Oracle(mb)
    for t in (3.0, 6.5, 12.0):
        ga.advance(t, DT), gb.advance(t, DT)
        oa.advance(t, DT), ob.advance(t, DT)
    assert rel(ga.voltage(), oa.voltage()) < 1e-6 and rel(gb.voltage(), ob.voltage()) < 1e-6
    check_spikes(ga, oa, 40), check_spikes(gb, ob, 12)
    ga.close(), gb.close()


def test_no_synapses_no_network(B, orc):
    m = W.random_model(11, n_cells=4, max_syn=0, n_conn=0, n_ext=0, t_end=5.0)
    assert m["n_syn"] == 0
    lockstep(B, orc, m, 100)


def test_chunked_advance_and_short_last_step(B, orc):
    m = W.random_model(2, n_cells=6, t_end=10.0)
    g, o = B.Model(m), orc.Oracle(m)
    for t in (1.0, 1.0125, 3.3, 3.3, 7.5, 10.0):            # non-multiples of dt, a zero-length call
        g.advance(t, DT)
        o.advance(t, DT)
        check_state(g, o, 1e-9, "t=%g" % t)
    assert g.time() == 10.0
    check_spikes(g, o, 6)
    assert tuple(g.probe(B.ARB_PROBE_NSTEPS)) == tuple(o.probe(orc.PROBE_NSTEPS))
    g.close()


def test_dt_can_change_between_calls(B, orc):
    m = W.random_model(6, n_cells=5, t_end=10.0)
    g, o = B.Model(m), orc.Oracle(m)
    for t, dt in ((2.0, 0.025), (4.0, 0.0125), (6.0, 0.05), (8.0, 0.025)):
        g.advance(t, dt)
        o.advance(t, dt)
        check_state(g, o, 1e-9, "t=%g" % t)
    check_spikes(g, o, 5)
    g.close()


def test_api_errors(B):
    m = W.random_model(3, n_cells=3)
    g = B.Model(m)
    for args in ((1.0, 0.0), (1.0, -1.0), (1.0, 50.0), (float("nan"), DT)):
        with pytest.raises(B.ArbError) as e:
            g.advance(*args)
        assert e.value.code == B.ARB_E_INVALID
    g.advance(1.0, DT)
    with pytest.raises(B.ArbError):
        g.advance(0.5, DT)
    import ctypes as C
    out = np.empty(3)
    assert B.lib().arb_voltage(g._h, out.ctypes.data, 3) == B.ARB_E_INVALID
    assert b"mismatch" in B.lib().arb_last_error(g._h)
    g.close()


def test_spike_buffer_cap_and_order(B, orc):
    m = W.config1(n_cells=30, t_end=100.0)
    g, o = run_both(B, orc, m, 100.0)
    n = B.lib().arb_spikes(g._h, None, None, 0)
    assert n == len(o.spikes()[0]) and n > 5
    cell, t = np.full(3, -1, np.int64), np.zeros(3)
    assert B.lib().arb_spikes(g._h, cell.ctypes.data, t.ctypes.data, 3) == n
    oc, ot = o.spikes()
    assert np.array_equal(cell, oc[:3]) and np.all(np.diff(t) >= 0) and np.allclose(t, ot[:3], atol=1e-9)
    g.close()


# ---------------------------------------------------------------------------------------------
# full-size configurations: the WHOLE network against the oracle, in the launch configuration
# bench.py times (one launch per grid step, groups with events first)
# ---------------------------------------------------------------------------------------------
FREE_RUN_TOL = 1e-6     # free-running V, gates over several hundred steps of a spiking network (R16/R17)


def expected_deliveries(m, spikes, t_end):
    """Events delivered before t_end: external ones plus (spike + delay) of every out-connection."""
    sc, st = spikes
    n = int(np.count_nonzero(m["ext_time"] < t_end))
    if len(sc) and m["n_conn"]:
        order = np.argsort(m["conn_src"], kind="stable")
        src, dly = m["conn_src"][order], m["conn_delay"][order]
        lo, hi = np.searchsorted(src, sc, "left"), np.searchsorted(src, sc, "right")
        for a, b, ts in zip(lo, hi, st):
            n += int(np.count_nonzero(ts + dly[a:b] < t_end))
    return n


def whole_network(B, orc, m, t_end, min_spikes=0, calls=1):
    import os
    g = B.Model(m)
    g.set_option(B.ARB_OPT_FUSED_STEPS, 1)
    g.set_option(B.ARB_OPT_HOT_FIRST, 1)
    o = orc.Oracle(m, threads=os.cpu_count() or 4)
    for i in range(calls):
        g.advance(t_end * (i + 1) / calls, m["dt"])
    o.advance(t_end, m["dt"])
    n = check_spikes(g, o, m["n_cells"])
    assert n >= min_spikes, n
    assert tuple(g.probe(B.ARB_PROBE_NSTEPS)) == tuple(o.probe(orc.PROBE_NSTEPS))
    assert g.stats()["events_delivered"] == expected_deliveries(m, o.spikes(), t_end)
    check_state(g, o, FREE_RUN_TOL, "t=%g" % t_end)
    st = g.stats()
    g.close()
    o.close()
    return n, st


def test_full_size_c3_whole_network(B, orc, layout):
    """configs[3] at its full 100,000 cells (5.05e7 CVs), driven, stated weights, three epochs (600 steps): every
    cell's V, m, h, n, g, the spikes, the sub-step count and the number of delivered events against the oracle
    on the whole network.  Then the same network with weights x 4 so that it fires within the first epoch and
    network events (5e6 connections, pool carry-over between epochs) are delivered in the second and third."""
    if layout != "default":
        pytest.skip("full size runs once, in the layout bench.py times")
    m = W.config3(t_end=15.0)
    n, st = whole_network(B, orc, m, 15.0, calls=3)
    assert st["classes"] == 1 and st["units"] == 0 and st["groups"] * 4 >= m["n_cells"] and st["group_ctas"] >= 148
    m["conn_weight"] = m["conn_weight"] * 4
    m["ext_weight"] = m["ext_weight"] * 4
    n, st = whole_network(B, orc, m, 15.0, min_spikes=10000)
    assert st["events_delivered"] > int(np.count_nonzero(m["ext_time"] < 15.0)) + 100000    # network events arrived


def test_full_size_c4_whole_network(B, orc, layout):
    """configs[4] at its full 50,000 cells (1.56e7 CVs, every tree different), two epochs."""
    if layout != "default":
        pytest.skip("full size runs once, in the layout bench.py times")
    m = W.config4(t_end=10.0)
    whole_network(B, orc, m, 10.0, calls=2)


def test_full_size_c1_whole_run(B, orc, layout):
    """configs[1] at full size for its whole 200 ms (8,000 steps): the ring spike travels through 39 cells."""
    if layout != "default":
        pytest.skip("full size runs once, in the layout bench.py times")
    m = W.config1()
    n, _ = whole_network(B, orc, m, 200.0, min_spikes=30)


def test_full_size_c2_100ms(B, orc, layout):
    """configs[2] at full size (10,000 cells, 1e6 connections, 2e6 Poisson events per second): first 100 ms."""
    if layout != "default":
        pytest.skip("full size runs once, in the layout bench.py times")
    m = W.config2(t_end=100.0)
    whole_network(B, orc, m, 100.0)


# ---------------------------------------------------------------------------------------------
# other cell kinds: LIF cells and spike sources beside cable cells
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("seed", [0, 1, 2])
def test_mixed_cell_kinds_network(B, orc, seed):
    """Poisson spike sources drive LIF and cable cells which drive each other: identical spikes per cell (LIF and
    source spikes sit exactly on event / schedule times: equal to 1e-12), LIF potentials and cable voltages."""
    m = W.mixed_network(seed)
    g, o = run_both(B, orc, m, 60.0)
    n = check_spikes(g, o, m["n_cells"], tol=1e-9)
    kind = m["cell_kind"]
    gc, gt = g.spikes()
    assert n > 60 and np.count_nonzero(kind[gc] == 1) > 20 and np.count_nonzero(kind[gc] == 0) > 3
    src = np.flatnonzero(kind == 2)
    assert np.array_equal(np.sort(gt[np.isin(gc, src)]), np.sort(m["src_time"][m["src_time"] < 60.0]))
    gv, ov = g.voltage(), o.voltage()
    lif_cv = m["cv_off"][:-1][kind == 1]
    assert rel(gv[lif_cv], ov[lif_cv]) <= 1e-12
    assert rel(gv, ov) < 1e-6
    assert tuple(g.probe(B.ARB_PROBE_NSTEPS)) == tuple(o.probe(orc.PROBE_NSTEPS))
    g.close()


def test_mixed_cell_kinds_every_step(B, orc):
    lockstep(B, orc, W.mixed_network(3, n_cable=5, n_lif=6, n_src=3, t_end=15.0), 600)


def test_mixed_cell_kinds_launch_granularity_and_chunked_calls(B, orc):
    m = W.mixed_network(4)
    res = []
    for fused, cuts in ((0, (60.0,)), (1, (7.3, 20.0, 33.125, 60.0))):
        g = B.Model(m)
        g.set_option(B.ARB_OPT_FUSED_STEPS, fused)
        for t in cuts:
            g.advance(t, DT)
        res.append(g.spikes())
        g.close()
    assert np.array_equal(res[0][0], res[1][0]) and np.max(np.abs(res[0][1] - res[1][1])) < 1e-6


# ---------------------------------------------------------------------------------------------
# one network over several ranks: the ranks run one after the other on this GPU
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("n_ranks", [2, 3])
def test_sharded_network_equals_single_model_bit_for_bit(B, orc, n_ranks):
    """Cells split into contiguous ranges, connections by destination owner, spike blocks exchanged once per epoch
    (arb_spike_block / arb_apply_spike_blocks): the same bits as one model advanced with the same calls, and the
    oracle's spikes."""
    from paper_1901_07454_b200 import sharded as S
    m = W.config3(n_cells=90, t_end=40.0)
    m["conn_weight"] = m["conn_weight"] * 4
    m["ext_weight"] = m["ext_weight"] * 4
    grp = S.LocalGroup(B, m, n_ranks)
    single = B.Model(m)
    es = S.epoch_steps(float(np.min(m["conn_delay"])), DT)
    k = 0
    while k * DT < 40.0:
        k += es
        t = min(40.0, k * DT)
        grp.advance(t, DT)
        single.advance(t, DT)
    assert np.array_equal(grp.gather(lambda g: g.voltage()), single.voltage())
    assert np.array_equal(grp.gather(lambda g: g.syn_g()), single.syn_g())
    for a, b in zip(grp.gather(lambda g: np.stack(g.gates(), 1)).T, single.gates()):
        assert np.array_equal(a, b)
    gc, gt = grp.spikes()
    sc, st = single.spikes()
    assert np.array_equal(gc, sc) and np.array_equal(gt, st) and len(sc) > 20
    assert sum(s.model.stats()["events_delivered"] for s in grp.ranks) == single.stats()["events_delivered"]
    o = orc.Oracle(m, threads=4)
    o.advance(40.0, DT)
    check_spikes(single, o, 90)
    grp.close(), single.close()


def test_sharded_overlapped_exchange_equals_single_model(B):
    """overlap=True: exchange epochs of half the minimum delay, the spikes of half-epoch h applied after half-epoch h + 1
    (the order a run takes whose all-gather is hidden behind the integration).  Same results as the
    single model, whatever the call pattern."""
    from paper_1901_07454_b200 import sharded as S
    m = W.config3(n_cells=90, t_end=40.0)
    m["conn_weight"] = m["conn_weight"] * 4
    m["ext_weight"] = m["ext_weight"] * 4
    grp = S.LocalGroup(B, m, 3, overlap=True)
    assert S.exchange_steps(grp.min_delay, DT, True) == S.epoch_steps(grp.min_delay, DT) // 2
    single = B.Model(m)
    for t in (13.0, 13.4, 40.0):                  # calls that end inside an epoch, too
        grp.advance(t, DT)
        single.advance(t, DT)
    # the shards restart their time grid at every half-epoch (t0 + k dt with another t0), the single model at every call:
    # event times inside a step differ by an ulp, so equality holds to rounding, not bit for bit
    assert rel(grp.gather(lambda g: g.voltage()), single.voltage()) < 1e-9
    assert rel(grp.gather(lambda g: g.syn_g()), single.syn_g()) < 1e-9
    gc, gt = grp.spikes()
    sc, st = single.spikes()
    assert np.array_equal(gc, sc) and np.max(np.abs(gt - st)) < 1e-9 and len(sc) > 20
    assert sum(s.model.stats()["events_delivered"] for s in grp.ranks) == single.stats()["events_delivered"]
    grp.close(), single.close()


def test_sharded_heterogeneous_network(B, orc):
    """configs[4] cut over two ranks (forests and groups on both): spikes against the oracle."""
    from paper_1901_07454_b200 import sharded as S
    m = W.config4(n_cells=80, t_end=30.0)
    grp = S.LocalGroup(B, m, 2)
    grp.advance(30.0, DT)
    o = orc.Oracle(m, threads=4)
    o.advance(30.0, DT)
    gc, gt = grp.spikes()
    oc, ot = o.spikes()
    assert np.array_equal(np.bincount(gc, minlength=80), np.bincount(oc, minlength=80)) and len(oc) > 10
    gi, oi = np.lexsort((gt, gc)), np.lexsort((ot, oc))
    assert np.max(np.abs(gt[gi] - ot[oi])) <= 1e-3
    assert rel(grp.gather(lambda g: g.voltage()), o.voltage()) < 1e-6
    grp.close()


# ---------------------------------------------------------------------------------------------
# capacities and error paths (include/arbb200.h "Capacities")
# ---------------------------------------------------------------------------------------------
def _firing_net(t_end=40.0):
    m = W.config1(n_cells=30, t_end=t_end)
    return m


def test_spike_buffer_overflow_is_reported(B, orc):
    m = _firing_net()
    m["cap_spikes"] = 2
    g = B.Model(m)
    with pytest.raises(B.ArbError) as e:
        g.advance(40.0, DT)
    assert e.value.code == B.ARB_E_OVERFLOW and "cap_spikes" in str(e.value)
    with pytest.raises(B.ArbError) as e:          # unusable afterwards, same code
        g.advance(41.0, DT)
    assert e.value.code == B.ARB_E_OVERFLOW
    g.close()


def test_spike_buffer_is_drained_between_calls(B, orc):
    """A device spike buffer of 2 entries is enough when it is drained often enough: the history lives in
    host memory, arb_spikes stays cumulative, arb_clear_spikes empties it."""
    m = _firing_net()
    m["cap_spikes"] = 2
    g, o = B.Model(m), orc.Oracle(m)
    for k in range(1, 9):
        g.advance(5.0 * k, DT)
    o.advance(40.0, DT)
    assert check_spikes(g, o, 30) >= 6
    g.clear_spikes()
    assert len(g.spikes()[0]) == 0
    g.close()


def test_event_pool_overflow_is_reported(B, orc):
    m = W.config3(n_cells=60, t_end=30.0)
    m["conn_weight"] = m["conn_weight"] * 4
    m["ext_weight"] = m["ext_weight"] * 4
    m["cap_events"] = 8
    g = B.Model(m)
    with pytest.raises(B.ArbError) as e:
        g.advance(30.0, DT)
    assert e.value.code == B.ARB_E_OVERFLOW and "cap_events" in str(e.value) and "event pool" in str(e.value)
    g.close()
    # the default capacity takes the same run
    del m["cap_events"]
    g, o = run_both(B, orc, m, 30.0)
    assert check_spikes(g, o, 60) > 5
    g.close()


def test_long_delays_fit_the_default_pool(B, orc):
    """Delays of 40 ms against 5 ms inter-spike intervals: several events per connection in flight."""
    m = W.config1(n_cells=8, t_end=150.0)
    m["conn_delay"] = np.full(m["n_conn"], 40.0)
    m["clamp_cell"], m["clamp_cv"] = np.array([0]), np.array([0], np.int32)
    m["clamp_t0"], m["clamp_t1"], m["clamp_amp"] = np.array([0.0]), np.array([150.0]), np.array([0.2])
    m = W.finalize(m)
    g, o = run_both(B, orc, m, 150.0)
    assert check_spikes(g, o, 8) > 10
    g.close()


def test_divergence_is_reported(B):
    """dt = 1 ms on the HH soma: the explicit membrane currents (reading R1) blow up; the oracle ends in NaN
    too.  The library reports it instead of returning garbage."""
    g = B.Model(W.config0())
    with pytest.raises(B.ArbError) as e:
        g.advance(100.0, 1.0)
    assert e.value.code == B.ARB_E_DIVERGED
    g.close()


def test_fp64_peak_measurement(B):
    """arb_fp64_peak: the DFMA rate of the device lies between a tenth of and the nominal fp64 peak
    (148 SMs x 64 DFMA/clk x < 2.2 GHz = 2.1e13, B200_PROFILING.md unit counts)."""
    import torch
    rate, ms = B.arb_fp64_peak(torch.cuda.current_stream().cuda_stream)
    assert 2e12 < rate < 2.2e13 and ms > 0
