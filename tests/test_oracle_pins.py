"""Pins of the CPU oracle against things other than itself.

Each test names the passage of PAPER.md whose implementation it pins.  None of these needs a GPU.
"""
import os

import numpy as np
import pytest

from paper_1901_07454_b200 import workloads as W

DT = 0.025
GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _dense_system(parent, area, cm, rax, v, i_memb, delta):
    """PAPER.md:154 written as a dense matrix: (diag(c/dt) + weighted Laplacian) V' = c/dt V - I."""
    n = len(parent)
    A = np.zeros((n, n))
    c = cm * area * 1e-5
    for i in range(n):
        A[i, i] += c[i] / delta
    for i in range(1, n):
        s = 1.0 / rax[i]
        p = parent[i]
        A[i, i] += s
        A[p, p] += s
        A[i, p] -= s
        A[p, i] -= s
    return A, c / delta * v - i_memb


# ---------------------------------------------------------------------------------------------
# P1 Hines solve == LAPACK dense solve, P2 assembly structure
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("kind", ["random", "chain", "star", "binary", "bushy"])
def test_p1_hines_vs_dense_lu(orc, kind):
    rng = np.random.default_rng(11)
    for trial in range(40):
        n = int(rng.integers(1, 65))
        parent = W.random_parent(rng, n, kind)
        area, cm = rng.uniform(10, 800, n), rng.uniform(0.5, 2, n)
        rax = rng.uniform(0.05, 60, n)
        v, im = rng.uniform(-80, 40, n), rng.uniform(-2, 2, n)
        delta = float(rng.choice([0.025, 0.0125, 1e-3, 0.2, 3e-7]))
        d, u, rhs = orc.assemble(parent, area, cm, rax, v, im, delta)
        x = orc.hines_solve(parent, d, u, rhs)
        A, b = _dense_system(parent, area, cm, rax, v, im, delta)
        ref = np.linalg.solve(A, b)
        assert np.max(np.abs(x - ref)) <= 1e-13 * np.max(np.abs(ref)), (kind, n, trial)


def test_p2_assembly_symmetric_diagonally_dominant(orc):
    rng = np.random.default_rng(12)
    for trial in range(30):
        n = int(rng.integers(2, 65))
        parent = W.random_parent(rng, n, "random")
        area, cm, rax = rng.uniform(10, 800, n), rng.uniform(0.5, 2, n), rng.uniform(0.05, 60, n)
        v, im = rng.uniform(-80, 40, n), rng.uniform(-2, 2, n)
        delta = 0.025
        d, u, rhs = orc.assemble(parent, area, cm, rax, v, im, delta)
        assert u[0] == 0.0 and np.all(u[1:] < 0)
        # row sums: d_i - sum|offdiag| = C_i/delta  (strict diagonal dominance)
        off = np.zeros(n)
        for i in range(1, n):
            off[i] += -u[i]
            off[parent[i]] += -u[i]
        c_over_dt = cm * area * 1e-5 / delta
        assert np.allclose(d - off, c_over_dt, rtol=1e-13, atol=0)
        # u_i = -1/raxial_i : doubling one resistance halves exactly that coupling
        rax2 = rax.copy()
        rax2[n - 1] *= 2
        _, u2, _ = orc.assemble(parent, area, cm, rax2, v, im, delta)
        assert u2[n - 1] == pytest.approx(u[n - 1] / 2, rel=1e-15)
        # rhs is linear in I with coefficient -1 and in V with coefficient C/dt
        _, _, rhs2 = orc.assemble(parent, area, cm, rax, v, im + 1.0, delta)
        assert np.allclose(rhs - rhs2, 1.0, rtol=0, atol=1e-12)
        _, _, rhs3 = orc.assemble(parent, area, cm, rax, v + 1.0, im, delta)
        assert np.allclose(rhs3 - rhs, c_over_dt, rtol=1e-9)


# ---------------------------------------------------------------------------------------------
# P3 closed-form steady state of a passive unbranched cable
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("n", [1, 2, 7, 24])
def test_p3_passive_cable_steady_state(orc, n):
    g_pas, area, rax, e, i_inj = 1e-4, 100.0, 5.0, -65.0, 0.02
    m = W.passive_cable(n, g_pas=g_pas, area=area, rax=rax, e_pas=e, i_inj=i_inj, t_end=600.0)
    o = orc.Oracle(m)
    o.advance(600.0, DT)          # tau_m = C/G = 10 ms -> exp(-60) left
    v = o.voltage()
    G, s = g_pas * area * 1e-2, 1.0 / rax
    if n == 1:
        ref = np.array([e + i_inj / G])
    else:
        kappa = np.arccosh(1 + G / (2 * s))
        i = np.arange(n)
        ref = e + i_inj * np.cosh(kappa * (n - 0.5 - i)) / (2 * s * np.sinh(kappa * n) * np.sinh(kappa / 2))
    assert np.max(np.abs(v - ref)) <= 1e-9
    # sign (R8): positive clamp amplitude depolarises
    assert np.all(v > e)


def test_p3_converges_to_continuum_cable(orc):
    """First-order convergence (PAPER.md:121 'first-order approximation for the axial current
    flux') to V(x) = E + I r_a lam cosh((L-x)/lam)/sinh(L/lam)."""
    L, d, g_pas, e, i_inj = 1000.0, 1.0, 1e-3, -65.0, 0.05
    r_a = W.seg_resistance(1.0, d)               # MOhm per um
    g_m = g_pas * np.pi * d * 1e-2               # uS per um
    lam = 1.0 / np.sqrt(r_a * g_m)
    errs = []
    for n in (20, 40, 80):
        seg = L / n
        m = W.passive_cable(n, g_pas=g_pas, area=np.pi * d * seg, rax=W.seg_resistance(seg, d),
                            e_pas=e, i_inj=i_inj, t_end=30.0)
        o = orc.Oracle(m)
        o.advance(30.0, 0.005)                   # tau_m = 1 ms
        x = (np.arange(n) + 0.5) * seg
        ref = e + i_inj * r_a * lam * np.cosh((L - x) / lam) / np.sinh(L / lam)
        errs.append(np.max(np.abs(o.voltage() - ref)))
    assert errs[0] > errs[1] > errs[2]
    assert 1.6 < errs[0] / errs[1] < 4.5 and 1.6 < errs[1] / errs[2] < 4.5


# ---------------------------------------------------------------------------------------------
# P4 per-step decay of the eigenmodes of the linear part            (R1)
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("k", [0, 1, 3, 11])
def test_p4_eigenmode_decay(orc, k):
    n, g_pas, area, rax, cm, e = 12, 2e-4, 150.0, 3.0, 1.3, -65.0
    i = np.arange(n)
    mode = np.cos(np.pi * k * (i + 0.5) / n)
    m = W.passive_cable(n, g_pas=g_pas, area=area, rax=rax, cm=cm, e_pas=e, vinit=e + mode)
    o = orc.Oracle(m)
    nsteps = 50
    o.advance(nsteps * DT, DT)
    G, C, s = g_pas * area * 1e-2, cm * area * 1e-5, 1.0 / rax
    lam_k = 2 * s * (1 - np.cos(np.pi * k / n))
    rho = (1 - DT * G / C) / (1 + DT * lam_k / C)     # explicit leak, implicit axial (R1)
    assert np.max(np.abs(o.voltage() - (e + rho ** nsteps * mode))) <= 2e-12


# ---------------------------------------------------------------------------------------------
# P5 charge / current balance, also at branch points                (eq 2a)
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("seed", [1, 2, 3])
def test_p5_current_balance(orc, seed):
    m = W.random_model(seed, n_cells=4, n_ext=0, n_conn=0, t_end=5.0)
    o = orc.Oracle(m)
    o.advance(1.0, DT)                     # get away from the initial state
    for _ in range(3):
        v0 = o.voltage()
        cur = [o.currents(c) for c in range(m["n_cells"])]
        t0 = o.time()
        o.advance(t0 + DT, DT)
        v1 = o.voltage()
        for c in range(m["n_cells"]):
            a, b = m["cv_off"][c], m["cv_off"][c + 1]
            C = m["cv_cm"][a:b] * m["cv_area"][a:b] * 1e-5
            par = m["cv_parent"][a:b]
            dv = (v1[a:b] - v0[a:b]) / DT
            scale = np.max(np.abs(C * dv)) + np.max(np.abs(cur[c])) + 1e-3
            # whole cell: axial terms cancel
            assert abs(np.sum(C * dv) + np.sum(cur[c])) <= 1e-11 * scale * (b - a)
            # per CV
            res = C * dv + cur[c]
            for i in range(1, b - a):
                s = 1.0 / m["cv_raxial"][a + i]
                flow = s * (v1[a + i] - v1[a + par[i]])
                res[i] += flow
                res[par[i]] -= flow
            assert np.max(np.abs(res)) <= 1e-10 * scale


# ---------------------------------------------------------------------------------------------
# P6 / P7 HH constants, fixed point, removable singularities        (R5)
# ---------------------------------------------------------------------------------------------
def _gold(name):
    out = {}
    for line in open(os.path.join(GOLD, name)):
        if line.strip() and not line.startswith("#"):
            k, v, tol = line.split()
            out[k] = (float(v), float(tol))
    return out


def test_p6_hh_textbook_values(orc):
    g = _gold("hh_rest_m65.txt")
    r = orc.hh_rates(-65.0)
    vals = dict(alpha_m=r[0], beta_m=r[1], alpha_h=r[2], beta_h=r[3], alpha_n=r[4], beta_n=r[5],
                m_inf=r[0] / (r[0] + r[1]), h_inf=r[2] / (r[2] + r[3]), n_inf=r[4] / (r[4] + r[5]))
    for k, (v, tol) in g.items():
        assert abs(vals[k] - v) <= tol, k
    # initial gates (R4) are the steady state at V_init
    m = W.random_model(5, n_cells=2, vinit=False, n_ext=0, n_conn=0)
    o = orc.Oracle(m)
    hm, hh, hn = o.gates()
    has = m["hh_gnabar"] != 0
    assert has.any()
    assert np.allclose(hm[has], vals["m_inf"], atol=1e-15) and np.allclose(hh[has], vals["h_inf"], atol=1e-15)
    assert np.allclose(hn[has], vals["n_inf"], atol=1e-15) and np.all(hm[~has] == 0)


def _single_hh(vinit, amp=0.0, t0=0.0, t1=0.0, t_end=50.0):
    m = dict(n_cells=1, cv_off=[0, 1], cv_parent=[-1], cv_area=[500.0], cv_cm=[1.0], cv_raxial=[1.0],
             cv_vinit=[vinit], hh_gnabar=[W.GNABAR], hh_gkbar=[W.GKBAR], hh_gl=[W.GL], t_end=t_end)
    if amp:
        m.update(clamp_cell=[0], clamp_cv=[0], clamp_t0=[t0], clamp_t1=[t1], clamp_amp=[amp])
    return W.finalize(m)


def test_p6_rest_potential_is_a_fixed_point(orc):
    def i_ion(v):
        r = orc.hh_rates(v)
        mi, hi, ni = r[0] / (r[0] + r[1]), r[2] / (r[2] + r[3]), r[4] / (r[4] + r[5])
        return W.GNABAR * mi ** 3 * hi * (v - W.ENA) + W.GKBAR * ni ** 4 * (v - W.EK) + W.GL * (v - W.EL)
    lo, hi = -70.0, -60.0
    assert i_ion(lo) < 0 < i_ion(hi)
    for _ in range(200):
        mid = 0.5 * (lo + hi)
        lo, hi = (mid, hi) if i_ion(mid) < 0 else (lo, mid)
    vrest = 0.5 * (lo + hi)
    assert abs(vrest - (-64.974)) < 2e-3                     # ~ -64.974 mV
    o = orc.Oracle(_single_hh(vrest))
    prev = vrest
    for _ in range(20):                                       # 20 x 100 steps
        o.advance(o.time() + 100 * DT, DT)
        v = o.voltage()[0]
        assert abs(v - prev) <= 100 * 1e-12
        prev = v
    assert abs(prev - vrest) < 1e-9
    # from -65 mV it relaxes towards that root and fires no spike
    o = orc.Oracle(_single_hh(-65.0))
    o.advance(100.0, DT)
    assert abs(o.voltage()[0] - vrest) < 1e-3 and len(o.spikes()[1]) == 0


def test_p7_exprelr_removable_singularity(orc):
    assert orc.exprelr(0.0) == 1.0
    assert orc.hh_rates(-40.0)[0] == 1.0 and orc.hh_rates(-55.0)[4] == 0.1
    for v0, idx in ((-40.0, 0), (-55.0, 4)):
        a, b, c = (orc.hh_rates(v0 + e)[idx] for e in (-1e-9, 0.0, 1e-9))
        assert abs(a - b) < 1e-9 and abs(c - b) < 1e-9 and a < b < c   # alpha increases with V
    # agrees with the textbook form away from the singularity
    for v in (-80.0, -41.0, -39.0, 0.0, 30.0):
        assert orc.hh_rates(v)[0] == pytest.approx(0.1 * (v + 40) / (1 - np.exp(-(v + 40) / 10)), rel=1e-13)
        assert orc.hh_rates(v)[4] == pytest.approx(0.01 * (v + 55) / (1 - np.exp(-(v + 55) / 10)), rel=1e-13)


# ---------------------------------------------------------------------------------------------
# P8 exponential synapse: decay and event delivery inside a step     (R7, R9)
# ---------------------------------------------------------------------------------------------
def _one_cv_syn(ext_time, ext_w, tau=2.0, e=0.0, t_end=10.0):
    m = dict(n_cells=1, cv_off=[0, 1], cv_parent=[-1], cv_area=[400.0], cv_cm=[1.0], cv_raxial=[1.0],
             pas_g=[1e-4], pas_e=[-65.0], syn_off=[0, 1], syn_cv=[0], syn_tau=[tau], syn_e=[e],
             ext_cell=np.zeros(len(ext_time), np.int64), ext_syn=np.zeros(len(ext_time), np.int32),
             ext_time=ext_time, ext_weight=ext_w, t_end=t_end)
    return W.finalize(m)


def test_p8_expsyn_decay_and_split_step(orc):
    w, tau = 0.013, 2.0
    o = orc.Oracle(_one_cv_syn([0.0], [w], tau))
    for k in (1, 10, 400):
        o.advance(k * DT, DT)
        assert o.syn_g()[0] == pytest.approx(w * np.exp(-k * DT / tau), rel=(k + 2) * 2.3e-16)
    # event strictly inside a step: exact decay from the event time (the step is split there)
    e = 3 * DT + 0.0071
    o = orc.Oracle(_one_cv_syn([e], [w], tau))
    o.advance(3 * DT, DT)
    assert o.syn_g()[0] == 0.0
    o.advance(4 * DT, DT)
    assert o.syn_g()[0] == pytest.approx(w * np.exp(-(4 * DT - e) / tau), rel=1e-15)
    assert tuple(o.probe(orc.PROBE_NSTEPS)) == (4.0, 5.0)        # one extra sub-step
    # two events on the same synapse at the same time add up; an event on a grid point is
    # delivered at the start of that step without a split
    o = orc.Oracle(_one_cv_syn([2 * DT, 2 * DT], [w, 2 * w], tau))
    o.advance(3 * DT, DT)
    assert o.syn_g()[0] == pytest.approx(3 * w * np.exp(-DT / tau), rel=1e-15)
    assert tuple(o.probe(orc.PROBE_NSTEPS)) == (3.0, 3.0)
    # synaptic current depolarises towards e (R7: I = g (V - e), enters eq 2a with a minus sign)
    assert o.voltage()[0] > -65.0


# ---------------------------------------------------------------------------------------------
# P9 the splitting integrator against an independent ODE solver
# ---------------------------------------------------------------------------------------------
def test_p9_first_order_convergence_to_solve_ivp(orc):
    from scipy.integrate import solve_ivp
    amp, t0, area = 0.08, 2.0, 500.0
    C = 1.0 * area * 1e-5

    def rates(v):           # textbook form, written independently of the oracle
        am = 0.1 * (v + 40) / (1 - np.exp(-(v + 40) / 10))
        bm = 4 * np.exp(-(v + 65) / 18)
        ah = 0.07 * np.exp(-(v + 65) / 20)
        bh = 1 / (1 + np.exp(-(v + 35) / 10))
        an = 0.01 * (v + 55) / (1 - np.exp(-(v + 55) / 10))
        bn = 0.125 * np.exp(-(v + 65) / 80)
        return am, bm, ah, bh, an, bn

    def f(t, y):
        v, m, h, n = y
        am, bm, ah, bh, an, bn = rates(v)
        dens = W.GNABAR * m ** 3 * h * (v - W.ENA) + W.GKBAR * n ** 4 * (v - W.EK) + W.GL * (v - W.EL)
        inj = amp if t >= t0 else 0.0
        return [(-dens * area * 1e-2 + inj) / C, am * (1 - m) - bm * m, ah * (1 - h) - bh * h,
                an * (1 - n) - bn * n]

    am, bm, ah, bh, an, bn = rates(-65.0)
    y0 = [-65.0, am / (am + bm), ah / (ah + bh), an / (an + bn)]
    up = lambda t, y: y[0] - W.THRESHOLD
    up.direction = 1
    s1 = solve_ivp(f, (0, t0), y0, rtol=1e-11, atol=1e-13, method="LSODA")
    s2 = solve_ivp(f, (t0, 30.0), s1.y[:, -1], rtol=1e-11, atol=1e-13, method="LSODA", events=up)
    ref = s2.t_events[0]
    assert len(ref) >= 2
    errs = []
    for dt in (0.02, 0.01, 0.005):
        o = orc.Oracle(_single_hh(-65.0, amp, t0, 1e9, 30.0))
        o.advance(30.0, dt)
        ts = o.spikes()[1]
        assert len(ts) == len(ref)
        errs.append(abs(ts[0] - ref[0]))
    assert errs[0] < 0.2
    assert 1.7 < errs[0] / errs[1] < 2.3 and 1.7 < errs[1] / errs[2] < 2.3


# ---------------------------------------------------------------------------------------------
# P10 ordering invariance                                            ("appropriate numbering")
# ---------------------------------------------------------------------------------------------
def _renumber_cvs(m, rng):
    """Another valid topological numbering of every cell's CVs (root stays 0)."""
    m = dict(m)
    perm_all = np.empty(m["n_cv"], np.int64)       # new global index -> old global index
    new_parent = np.empty(m["n_cv"], np.int32)
    syn_cv = m["syn_cv"].copy()
    for c in range(m["n_cells"]):
        a, b = m["cv_off"][c], m["cv_off"][c + 1]
        par = m["cv_parent"][a:b]
        n = b - a
        kids = [[] for _ in range(n)]
        for i in range(1, n):
            kids[par[i]].append(i)
        order, front = [], [0]
        while front:                                # random frontier expansion
            j = front.pop(int(rng.integers(len(front))))
            order.append(j)
            front += kids[j]
        order = np.array(order)
        inv = np.empty(n, np.int64)
        inv[order] = np.arange(n)
        perm_all[a:b] = a + order
        new_parent[a:b] = [-1 if par[o] < 0 else inv[par[o]] for o in order]
        s0, s1 = m["syn_off"][c], m["syn_off"][c + 1]
        syn_cv[s0:s1] = inv[m["syn_cv"][s0:s1]]
        m["clamp_cv"] = np.where(m["clamp_cell"] == c, inv[np.minimum(m["clamp_cv"], n - 1)], m["clamp_cv"]).astype(np.int32)
        if m["det_cv"] is not None:
            m["det_cv"] = m["det_cv"].copy()
            m["det_cv"][c] = inv[m["det_cv"][c]]
    for k in ("cv_area", "cv_cm", "cv_raxial", "cv_vinit", "hh_gnabar", "hh_gkbar", "hh_gl", "pas_g", "pas_e"):
        if m[k] is not None:
            m[k] = m[k][perm_all]
    m["cv_parent"], m["syn_cv"] = new_parent, syn_cv
    return W.finalize(m), perm_all


def _permute_cells(m, perm):
    """Cell new index i is old cell perm[i]; connections / events / clamps follow."""
    inv = np.empty(len(perm), np.int64)
    inv[perm] = np.arange(len(perm))
    out = W.take_cells(m, perm)
    out["conn_src"], out["conn_dst"] = inv[m["conn_src"]], inv[m["conn_dst"]]
    for k in ("conn_syn", "conn_delay", "conn_weight"):
        out[k] = m[k]
    return W.finalize(out)


def _run(orc, m, t_end):
    o = orc.Oracle(m)
    o.advance(t_end, m["dt"])
    return o.voltage(), o.spikes()


def test_p10_cv_renumbering_and_cell_permutation(orc):
    rng = np.random.default_rng(5)
    m = W.random_model(8, n_cells=6, t_end=20.0)
    v, (sc, st) = _run(orc, m, 20.0)
    assert len(st) > 0
    m2, perm = _renumber_cvs(m, rng)
    v2, (sc2, st2) = _run(orc, m2, 20.0)
    assert np.array_equal(sc, sc2)
    assert np.max(np.abs(st - st2)) <= 1e-9
    assert np.max(np.abs(v2 - v[perm])) <= 1e-9 * max(1, np.max(np.abs(v)))
    # over a single step the agreement is at rounding level
    v1, _ = _run(orc, m, DT)
    v1b, _ = _run(orc, m2, DT)
    assert np.max(np.abs(v1b - v1[perm])) <= 1e-12 * 70
    # permuting the cells is bit-exact per cell
    cp = rng.permutation(m["n_cells"])
    m3 = _permute_cells(m, cp)
    v3, (sc3, st3) = _run(orc, m3, 20.0)
    for i, c in enumerate(cp):
        assert np.array_equal(v3[m3["cv_off"][i]:m3["cv_off"][i + 1]], v[m["cv_off"][c]:m["cv_off"][c + 1]])
    assert np.array_equal(np.sort(st3), np.sort(st))


# ---------------------------------------------------------------------------------------------
# P11 network path
# ---------------------------------------------------------------------------------------------
def test_p11_event_time_is_spike_time_plus_delay(orc):
    """Two single-CV cells: A (HH, clamp) spikes at ts; B sees g jump by w at exactly ts+delay;
    a third connection with another delay / weight lands on B's second synapse."""
    tau = 3.0
    m = dict(n_cells=2, cv_off=[0, 1, 2], cv_parent=[-1, -1], cv_area=[500.0, 500.0], cv_cm=[1.0, 1.0],
             cv_raxial=[1.0, 1.0], hh_gnabar=[W.GNABAR, 0], hh_gkbar=[W.GKBAR, 0], hh_gl=[W.GL, 0],
             pas_g=[0, 1e-4], pas_e=[-65.0, -65.0], syn_off=[0, 0, 2], syn_cv=[0, 0],
             syn_tau=[tau, tau], syn_e=[0.0, 0.0],
             clamp_cell=[0], clamp_cv=[0], clamp_t0=[1.0], clamp_t1=[3.0], clamp_amp=[0.5],
             conn_src=[0, 0], conn_dst=[1, 1], conn_syn=[0, 1], conn_delay=[2.0 + 1 / 3, 4.7],
             conn_weight=[0.0004, 0.0009], t_end=12.0)
    m = W.finalize(m)
    o = orc.Oracle(m)
    o.advance(12.0, DT)
    sc, st = o.spikes()
    assert list(sc) == [0] and 1.0 < st[0] < 3.5
    g = o.syn_g()
    assert g[0] == pytest.approx(0.0004 * np.exp(-(12.0 - (st[0] + (2.0 + 1 / 3))) / tau), rel=1e-13)
    assert g[1] == pytest.approx(0.0009 * np.exp(-(12.0 - (st[0] + 4.7)) / tau), rel=1e-13)
    # nothing is delivered before its time
    o = orc.Oracle(m)
    te = st[0] + (2.0 + 1 / 3)
    k = int(np.floor(te / DT))
    o.advance(k * DT, DT)
    assert o.syn_g()[0] == 0.0
    o.advance((k + 1) * DT, DT)
    assert o.syn_g()[0] == pytest.approx(0.0004 * np.exp(-((k + 1) * DT - te) / tau), rel=1e-12)
    # the spike time is the linear interpolation of the crossing inside its step (R10)
    o = orc.Oracle(m)
    j = int(np.floor(st[0] / DT))
    o.advance(j * DT, DT)
    va = o.voltage()[0]
    o.advance((j + 1) * DT, DT)
    vb = o.voltage()[0]
    assert va < W.THRESHOLD <= vb
    assert st[0] == pytest.approx(j * DT + DT * (W.THRESHOLD - va) / (vb - va), abs=1e-12)


def test_p11_ring_invariant(orc):
    """PAPER.md:293 'trivial for the ring model': cells fire in index order, once per lap,
    successive lags >= delay."""
    n = 12
    m = W.config1(n_cells=n, t_end=140.0)
    o = orc.Oracle(m)
    o.advance(140.0, DT)
    sc, st = o.spikes()
    assert len(sc) >= n + 2                                 # more than one lap
    assert np.array_equal(sc, np.arange(len(sc)) % n)
    assert np.all(np.diff(st) >= 5.0)


# ---------------------------------------------------------------------------------------------
# P12 step splitting is continuous in the event time                 (R9)
# ---------------------------------------------------------------------------------------------
def test_p12_event_time_continuity_across_grid_point(orc):
    base = W.random_model(4, n_cells=2, n_ext=0, n_conn=0, n_clamp=0, t_end=2.0)
    res = []
    for shift in (-1e-9, 0.0, 1e-9):
        m = dict(base)
        cell = int(np.flatnonzero(np.diff(base["syn_off"]) > 0)[0])
        m.update(ext_cell=[cell], ext_syn=[0], ext_time=[40 * DT + shift], ext_weight=[0.03])
        m = W.finalize(m)
        o = orc.Oracle(m)
        o.advance(2.0, DT)
        res.append(o.voltage())
    assert np.max(np.abs(res[1] - base_run(orc, base))) > 1e-3          # the event matters
    assert np.max(np.abs(res[0] - res[1])) < 1e-7 and np.max(np.abs(res[2] - res[1])) < 1e-7


def base_run(orc, m):
    o = orc.Oracle(m)
    o.advance(2.0, DT)
    return o.voltage()


# ---------------------------------------------------------------------------------------------
# host logic: time grid, chunked advance, validation
# ---------------------------------------------------------------------------------------------
def test_chunked_advance_matches_single_call(orc):
    m = W.random_model(2, n_cells=6, t_end=10.0)
    v_ref, (_, st_ref) = _run(orc, m, 10.0)
    assert len(st_ref) > 0
    o = orc.Oracle(m)
    for t in (1.0, 1.0125, 3.3, 7.5, 10.0):                 # includes non-multiples of dt
        o.advance(t, DT)
    assert o.time() == 10.0
    st = o.spikes()[1]
    assert len(st) == len(st_ref)
    assert np.max(np.abs(o.voltage() - v_ref)) < 0.5        # shortened steps change the scheme at O(dt)
    o = orc.Oracle(m)
    for t in (2.5, 5.0, 7.5, 10.0):                         # multiples of dt: same grid up to rounding
        o.advance(t, DT)
    assert np.max(np.abs(o.voltage() - v_ref)) < 1e-8
    assert np.max(np.abs(o.spikes()[1] - st_ref)) < 1e-8
    assert o.probe(orc.PROBE_NSTEPS)[0] == 400


def test_validation_errors(orc):
    def bad(**kw):
        m = dict(W.random_model(3, n_cells=3))
        for k, v in kw.items():
            a = np.array(m[k], copy=True)
            a[v[0]] = v[1]
            m[k] = a
        with pytest.raises(orc.OracleError):
            orc.Oracle(W.finalize(m))
    bad(cv_parent=(0, 0))
    bad(cv_area=(1, -1.0))
    bad(cv_cm=(0, 0.0))
    bad(syn_tau=(0, 0.0))
    bad(conn_delay=(0, 0.0))
    bad(conn_src=(0, 99))
    bad(ext_time=(0, -1.0))
    bad(cv_area=(0, np.nan))
    m = W.random_model(3, n_cells=3)
    o = orc.Oracle(m)
    with pytest.raises(orc.OracleError):
        o.advance(1.0, 0.0)
    with pytest.raises(orc.OracleError):
        o.advance(1.0, 10.0)                                 # dt longer than the shortest delay
    o.advance(1.0, DT)
    with pytest.raises(orc.OracleError):
        o.advance(0.5, DT)


# ---------------------------------------------------------------------------------------------
# P13 synapse current I = g (V - e): magnitude and reversal potential   (eq 2a, R7)
# Mutations this pin kills (tests/test_oracle_mutations.py): `I += 0.5*g*(V-e)`, `I += g*(V+e)`.
# ---------------------------------------------------------------------------------------------
def _one_cv_syns(es, taus, area=400.0, g_pas=1e-4, e_pas=-65.0, vinit=-60.0):
    n = len(es)
    m = dict(n_cells=1, cv_off=[0, 1], cv_parent=[-1], cv_area=[area], cv_cm=[1.0], cv_raxial=[1.0],
             cv_vinit=[vinit], pas_g=[g_pas], pas_e=[e_pas], syn_off=[0, n], syn_cv=[0] * n,
             syn_tau=taus, syn_e=es, t_end=10.0)
    return W.finalize(m)


def test_p13_synapse_current_magnitude_and_reversal(orc):
    area, g_pas, e_pas, v0 = 400.0, 1e-4, -65.0, -60.0
    C, G = 1.0 * area * 1e-5, g_pas * area * 1e-2
    # one synapse held at a known conductance, reversal potential != 0: one step of eq 2a / PAPER.md:154
    for g, e in ((0.003, -20.0), (0.0007, 15.0), (0.002, -80.0)):
        o = orc.Oracle(_one_cv_syns([e], [2.0], vinit=v0))
        o.set_state(syn_g=[g])
        o.advance(DT, DT)
        ref = ((C / DT) * v0 - G * (v0 - e_pas) - g * (v0 - e)) / (C / DT)
        assert o.voltage()[0] == pytest.approx(ref, rel=1e-13)
        assert (o.voltage()[0] > v0 - DT / C * G * (v0 - e_pas)) == (e > v0)     # pulls towards e
    # two synapses with different reversal potentials on the same CV add up
    (g1, e1), (g2, e2) = (0.0021, -10.0), (0.0013, -75.0)
    o = orc.Oracle(_one_cv_syns([e1, e2], [2.0, 3.0], vinit=v0))
    o.set_state(syn_g=[g1, g2])
    o.advance(DT, DT)
    ref = ((C / DT) * v0 - G * (v0 - e_pas) - g1 * (v0 - e1) - g2 * (v0 - e2)) / (C / DT)
    assert o.voltage()[0] == pytest.approx(ref, rel=1e-13)
    # constant conductance (tau -> infinity): the steady state is the conductance-weighted mean
    g, e = 0.0025, -30.0
    o = orc.Oracle(_one_cv_syns([e], [1e15], vinit=v0))
    o.set_state(syn_g=[g])
    o.advance(40.0, DT)                                   # tau_m = C/(G+g) ~ 1.4 ms
    assert o.voltage()[0] == pytest.approx((G * e_pas + g * e) / (G + g), abs=1e-10)
    assert o.syn_g()[0] == pytest.approx(g, rel=1e-10)


# ---------------------------------------------------------------------------------------------
# P14 "the state variables are integrated with the updated voltage values"
# Mutation this pin kills: gate rates evaluated at V(t) instead of V'.
# ---------------------------------------------------------------------------------------------
def test_p14_gates_are_integrated_with_the_updated_voltage(orc):
    def rates(v):           # textbook form (as in P9), independent of the oracle
        return (0.1 * (v + 40) / (1 - np.exp(-(v + 40) / 10)), 4 * np.exp(-(v + 65) / 18),
                0.07 * np.exp(-(v + 65) / 20), 1 / (1 + np.exp(-(v + 35) / 10)),
                0.01 * (v + 55) / (1 - np.exp(-(v + 55) / 10)), 0.125 * np.exp(-(v + 65) / 80))

    def gates_after(v, x, delta):
        r = rates(v)
        out = []
        for k in range(3):
            a, b = r[2 * k], r[2 * k + 1]
            inf = a / (a + b)
            out.append(inf + (x[k] - inf) * np.exp(-delta * (a + b)))
        return np.array(out)

    area, amp, v0 = 500.0, 2.0, -52.0                     # large clamp: V' - V is several mV
    x0 = np.array([0.31, 0.42, 0.47])
    o = orc.Oracle(_single_hh(v0, amp, 0.0, 1e9))
    o.set_state(m=[x0[0]], h=[x0[1]], n=[x0[2]])
    o.advance(DT, DT)
    C = 1.0 * area * 1e-5
    dens = W.GNABAR * x0[0] ** 3 * x0[1] * (v0 - W.ENA) + W.GKBAR * x0[2] ** 4 * (v0 - W.EK) + W.GL * (v0 - W.EL)
    v1 = v0 + DT / C * (amp - dens * area * 1e-2)         # single CV: eq at PAPER.md:154 has no axial term
    assert v1 - v0 > 3.0
    assert o.voltage()[0] == pytest.approx(v1, rel=1e-13)
    got = np.array([g[0] for g in o.gates()])
    with_new, with_old = gates_after(v1, x0, DT), gates_after(v0, x0, DT)
    assert np.max(np.abs(with_new - with_old)) > 1e-6     # the pin has teeth
    assert np.max(np.abs(got - with_new)) <= 1e-13
    assert np.max(np.abs(got - with_old)) > 1e-6


# ---------------------------------------------------------------------------------------------
# P15 clamp window t0 <= t < t1, t = step start                             (R8; eq 2a's injected current)
# Mutation this pin kills: `t0 < t && t <= t1`.
# ---------------------------------------------------------------------------------------------
def test_p15_clamp_window_is_half_open_at_the_step_start(orc):
    area, g_pas, e_pas, amp = 300.0, 2e-4, -65.0, 0.05
    C, G = 1.0 * area * 1e-5, g_pas * area * 1e-2
    m = W.finalize(dict(n_cells=1, cv_off=[0, 1], cv_parent=[-1], cv_area=[area], cv_cm=[1.0], cv_raxial=[1.0],
                        pas_g=[g_pas], pas_e=[e_pas], clamp_cell=[0], clamp_cv=[0], clamp_t0=[5 * DT],
                        clamp_t1=[7 * DT], clamp_amp=[amp], t_end=1.0))
    o = orc.Oracle(m)
    v, seen = e_pas, []
    for k in range(10):                                   # step k starts at t = k * dt
        on = 5 <= k < 7
        v = v - DT / C * (G * (v - e_pas) - (amp if on else 0.0))
        o.advance((k + 1) * DT, DT)
        assert o.voltage()[0] == pytest.approx(v, rel=1e-14), k
        seen.append(o.voltage()[0])
    assert seen[4] == e_pas and seen[5] > e_pas           # exactly steps 5 and 6 see the current
    assert seen[6] - seen[5] > 0.5 * (seen[5] - seen[4]) and seen[7] < seen[6]


def test_ninth_spike_in_one_grid_step_is_an_error_not_a_drop(orc):
    """The oracle keeps at most 8 spikes of a cell per grid step; a ninth must be reported."""
    dt, nsub = 0.05, 24
    area, cm = 400.0, 1.0
    C = cm * area * 1e-5
    delta = dt / nsub
    g_pas = 0.9 * C / delta / (area * 1e-2)                # leak wipes 90% of (V - E) per sub-step
    w = 0.4 * C / delta / 65.0                              # a sub-step with g = w lifts V by ~0.4 mV
    t = 2 * dt + (np.arange(nsub - 1) + 1) * delta
    wt = np.where(np.arange(nsub - 1) % 2 == 0, w, -w)
    m = W.finalize(dict(n_cells=1, cv_off=[0, 1], cv_parent=[-1], cv_area=[area], cv_cm=[cm], cv_raxial=[1.0],
                        pas_g=[g_pas], pas_e=[-65.0], syn_off=[0, 1], syn_cv=[0], syn_tau=[1e9], syn_e=[0.0],
                        ext_cell=np.zeros(nsub - 1, np.int64), ext_syn=np.zeros(nsub - 1, np.int32), ext_time=t,
                        ext_weight=wt, threshold=-64.9, dt=dt, t_end=1.0))
    o = orc.Oracle(m)
    o.advance(2 * dt, dt)
    assert len(o.spikes()[1]) == 0
    with pytest.raises(orc.OracleError, match="more than 8 spikes"):
        o.advance(3 * dt, dt)
    # eight or fewer are kept: the same input cut after 8 upward crossings
    m2 = dict(m)
    keep = 2 * 8 - 1
    m2.update(ext_cell=m["ext_cell"][:keep], ext_syn=m["ext_syn"][:keep], ext_time=t[:keep], ext_weight=wt[:keep])
    o = orc.Oracle(W.finalize(m2))
    o.advance(3 * dt, dt)
    assert len(o.spikes()[1]) == 8


# ---------------------------------------------------------------------------------------------
# L1-L4 the conductance-linearised step (PAPER.md:152-156 with the membrane
# conductances on the diagonal).  Pinned like the explicit step: dense LU, closed forms, an ODE solver.
# ---------------------------------------------------------------------------------------------
def _lin(orc, m):
    o = orc.Oracle(m)
    o.set_linearised(True)
    return o


@pytest.mark.parametrize("seed", [1, 2, 3, 4])
def test_l1_linearised_step_vs_dense_lu(orc, seed):
    """One step of a random model (HH, passive, synapses with per-synapse e, clamps) against a dense solve of
    (diag(C/dt + g) + Laplacian) V' = C/dt V + sum g E + I_inj written out here."""
    m = W.random_model(seed, n_cells=4, n_conn=0, n_ext=0, t_end=5.0)
    rng = np.random.default_rng(seed)
    o = _lin(orc, m)
    g0 = rng.uniform(0.0, 0.004, m["n_syn"])
    o.set_state(syn_g=g0)
    v0, (hm, hh, hn) = o.voltage(), o.gates()
    o.advance(DT, DT)
    v1 = o.voltage()
    for c in range(m["n_cells"]):
        a, b = m["cv_off"][c], m["cv_off"][c + 1]
        n = b - a
        area = m["cv_area"][a:b]
        A, rhs = _dense_system(m["cv_parent"][a:b], area, m["cv_cm"][a:b], m["cv_raxial"][a:b], v0[a:b], np.zeros(n), DT)
        sc = area * 1e-2
        gna = m["hh_gnabar"][a:b] * hm[a:b] ** 3 * hh[a:b] * sc
        gk = m["hh_gkbar"][a:b] * hn[a:b] ** 4 * sc
        gl = m["hh_gl"][a:b] * sc
        gp = m["pas_g"][a:b] * sc
        g = gna + gk + gl + gp
        src = gna * m["hh_ena"] + gk * m["hh_ek"] + gl * m["hh_el"] + gp * m["pas_e"][a:b]
        for s in range(m["syn_off"][c], m["syn_off"][c + 1]):
            g[m["syn_cv"][s]] += g0[s]
            src[m["syn_cv"][s]] += g0[s] * m["syn_e"][s]
        for k in np.flatnonzero(m["clamp_cell"] == c):
            if m["clamp_t0"][k] <= 0.0 < m["clamp_t1"][k]:
                src[m["clamp_cv"][k]] += m["clamp_amp"][k]
        ref = np.linalg.solve(A + np.diag(g), rhs + src)
        assert np.max(np.abs(v1[a:b] - ref)) <= 1e-12 * np.max(np.abs(ref)), c


@pytest.mark.parametrize("k", [0, 1, 3, 11])
def test_l2_linearised_eigenmode_decay_is_fully_implicit(orc, k):
    """Passive chain: with the leak on the diagonal every mode decays by 1 / (1 + dt (G + lam_k) / C) per step
    (the explicit step of P4 has (1 - dt G / C) / (1 + dt lam_k / C))."""
    n, g_pas, area, rax, cm, e = 12, 2e-4, 150.0, 3.0, 1.3, -65.0
    i = np.arange(n)
    mode = np.cos(np.pi * k * (i + 0.5) / n)
    o = _lin(orc, W.passive_cable(n, g_pas=g_pas, area=area, rax=rax, cm=cm, e_pas=e, vinit=e + mode))
    nsteps = 50
    o.advance(nsteps * DT, DT)
    G, C, s = g_pas * area * 1e-2, cm * area * 1e-5, 1.0 / rax
    lam_k = 2 * s * (1 - np.cos(np.pi * k / n))
    rho = 1.0 / (1.0 + DT * (G + lam_k) / C)
    assert np.max(np.abs(o.voltage() - (e + rho ** nsteps * mode))) <= 2e-12
    rho_explicit = (1 - DT * G / C) / (1 + DT * lam_k / C)
    assert abs(rho - rho_explicit) > 1e-7                      # the two schemes differ: the pin tells them apart


def test_l3_linearised_steady_states(orc):
    """Steady states do not depend on the scheme: the cable of P3 and the conductance-weighted mean of P13."""
    n, g_pas, area, rax, e, i_inj = 7, 1e-4, 100.0, 5.0, -65.0, 0.02
    o = _lin(orc, W.passive_cable(n, g_pas=g_pas, area=area, rax=rax, e_pas=e, i_inj=i_inj, t_end=600.0))
    o.advance(600.0, DT)
    G, s = g_pas * area * 1e-2, 1.0 / rax
    kappa = np.arccosh(1 + G / (2 * s))
    i = np.arange(n)
    ref = e + i_inj * np.cosh(kappa * (n - 0.5 - i)) / (2 * s * np.sinh(kappa * n) * np.sinh(kappa / 2))
    assert np.max(np.abs(o.voltage() - ref)) <= 1e-9
    g, es, Gp = 0.0025, -30.0, 1e-4 * 400.0 * 1e-2
    o = _lin(orc, _one_cv_syns([es], [1e15], vinit=-60.0))
    o.set_state(syn_g=[g])
    o.advance(40.0, DT)
    assert o.voltage()[0] == pytest.approx((Gp * -65.0 + g * es) / (Gp + g), abs=1e-10)
    # one step of that CV by hand: V' = (C/dt V + G E + g e) / (C/dt + G + g)
    o = _lin(orc, _one_cv_syns([es], [2.0], vinit=-60.0))
    o.set_state(syn_g=[g])
    o.advance(DT, DT)
    C = 1.0 * 400.0 * 1e-5
    assert o.voltage()[0] == pytest.approx((C / DT * -60.0 + Gp * -65.0 + g * es) / (C / DT + Gp + g), rel=1e-14)


def test_l4_linearised_converges_to_the_same_ode(orc):
    """Single HH CV + current step against scipy: same spikes, first-order convergence (as P9), and it stays
    finite at dt = 1 ms where the explicit step diverges (tests/test_gpu_parity.py::test_divergence_is_reported)."""
    from scipy.integrate import solve_ivp
    amp, t0, area = 0.08, 2.0, 500.0
    C = 1.0 * area * 1e-5

    def f(t, y):
        v, m, h, n = y
        am = 0.1 * (v + 40) / (1 - np.exp(-(v + 40) / 10)); bm = 4 * np.exp(-(v + 65) / 18)
        ah = 0.07 * np.exp(-(v + 65) / 20); bh = 1 / (1 + np.exp(-(v + 35) / 10))
        an = 0.01 * (v + 55) / (1 - np.exp(-(v + 55) / 10)); bn = 0.125 * np.exp(-(v + 65) / 80)
        dens = W.GNABAR * m ** 3 * h * (v - W.ENA) + W.GKBAR * n ** 4 * (v - W.EK) + W.GL * (v - W.EL)
        return [(-dens * area * 1e-2 + (amp if t >= t0 else 0.0)) / C, am * (1 - m) - bm * m, ah * (1 - h) - bh * h,
                an * (1 - n) - bn * n]

    r = orc.hh_rates(-65.0)
    y0 = [-65.0, r[0] / (r[0] + r[1]), r[2] / (r[2] + r[3]), r[4] / (r[4] + r[5])]
    up = lambda t, y: y[0] - W.THRESHOLD
    up.direction = 1
    s1 = solve_ivp(f, (0, t0), y0, rtol=1e-11, atol=1e-13, method="LSODA")
    s2 = solve_ivp(f, (t0, 30.0), s1.y[:, -1], rtol=1e-11, atol=1e-13, method="LSODA", events=up)
    ref = s2.t_events[0]
    errs = []
    for dt in (0.02, 0.01, 0.005):
        o = _lin(orc, _single_hh(-65.0, amp, t0, 1e9, 30.0))
        o.advance(30.0, dt)
        ts = o.spikes()[1]
        assert len(ts) == len(ref)
        errs.append(abs(ts[0] - ref[0]))
    assert errs[0] < 0.2 and 1.6 < errs[0] / errs[1] < 2.4 and 1.6 < errs[1] / errs[2] < 2.4
    o = _lin(orc, W.config0())
    o.advance(100.0, 1.0)
    assert np.all(np.isfinite(o.voltage())) and np.all(np.abs(o.voltage()) < 200.0)


# ---------------------------------------------------------------------------------------------
# K1-K3 other cell kinds (reading R20): LIF cells and spike sources
# ---------------------------------------------------------------------------------------------
def _lif_net(ev_t, ev_w, t_end=50.0, **par):
    p = dict(W.LIF_DEFAULTS)
    p.update(par)
    m = dict(n_cells=1, cv_off=[0, 1], cv_parent=[-1], cv_area=[100.0], cv_cm=[1.0], cv_raxial=[1.0], cv_vinit=[p["lif_e_l"]],
             syn_off=[0, 1], syn_cv=[0], syn_tau=[2.0], syn_e=[0.0], cell_kind=[1],
             ext_cell=np.zeros(len(ev_t), np.int64), ext_syn=np.zeros(len(ev_t), np.int32), ext_time=ev_t, ext_weight=ev_w, t_end=t_end)
    for k, v in p.items():
        m[k] = [v]
    return W.finalize(m)


def test_k1_lif_closed_form_charging_spike_and_refractory(orc):
    tau, vth, cm, el, er, tref = 10.0, -50.0, 0.25, -65.0, -70.0, 6.0
    w, gap = 1.0, 1.3                                  # every event lifts V by w / C_m = 4 mV
    t = 0.7 + gap * np.arange(30)
    o = orc.Oracle(_lif_net(t, np.full(30, w), lif_tau_m=tau, lif_v_th=vth, lif_c_m=cm, lif_e_l=el, lif_e_r=er, lif_t_ref=tref))
    q = np.exp(-gap / tau)
    # geometric series until the threshold is reached
    k_spike = next(k for k in range(1, 31) if el + (w / cm) * (1 - q ** k) / (1 - q) >= vth)
    o.advance(t[k_spike - 2] + 0.01, DT)               # just after event k_spike - 1
    want = el + (w / cm) * (1 - q ** (k_spike - 1)) / (1 - q)
    assert o.voltage()[0] == pytest.approx(el + (want - el) * np.exp(-0.01 / tau), rel=1e-13)
    o.advance(50.0, DT)
    sc, st = o.spikes()
    assert st[0] == t[k_spike - 1]                     # the spike sits exactly on the event that crossed the threshold
    # events inside the refractory period are lost (four of them here); charging restarts from E_R at st + t_ref
    nxt = [x for x in t if x >= st[0] + tref]
    assert len([x for x in t if st[0] < x < st[0] + tref]) >= 4
    o2 = orc.Oracle(_lif_net(t, np.full(30, w), lif_tau_m=tau, lif_v_th=vth, lif_c_m=cm, lif_e_l=el, lif_e_r=er, lif_t_ref=tref))
    t_probe = 0.5 * (st[0] + tref + nxt[0])             # after the refractory period, before the next event
    o2.advance(t_probe, DT)
    assert o2.voltage()[0] == pytest.approx(el + (er - el) * np.exp(-(t_probe - (st[0] + tref)) / tau), rel=1e-13)
    v, tl = er, st[0] + tref
    second = None
    for x in nxt:
        v = el + (v - el) * np.exp(-(x - tl) / tau) + w / cm
        tl = x
        if v >= vth:
            second = x
            break
    assert second is not None and st[1] == second and len(st) >= 2
    assert np.all(np.diff(st) >= tref)


def test_k2_spike_sources_emit_their_schedule_and_drive_a_cable_cell(orc):
    """A source cell's spikes are its schedule; a connection source -> cable cell delivers g += w at t + delay."""
    sched = np.array([0.4, 3.3, 3.31, 7.0, 12.0, 19.5])   # 0.4 and 12.0 lie on grid points; 12.0 is the end of the run
    m = dict(n_cells=2, cv_off=[0, 1, 2], cv_parent=[-1, -1], cv_area=[100.0, 400.0], cv_cm=[1.0, 1.0], cv_raxial=[1.0, 1.0],
             pas_g=[0.0, 1e-4], pas_e=[-65.0, -65.0], syn_off=[0, 0, 1], syn_cv=[0], syn_tau=[3.0], syn_e=[0.0],
             cell_kind=[2, 0], src_off=[0, 6, 6], src_time=sched,
             conn_src=[0], conn_dst=[1], conn_syn=[0], conn_delay=[1.25], conn_weight=[0.0002], t_end=12.0)
    m = W.finalize(m)
    o = orc.Oracle(m)
    o.advance(12.0, DT)
    sc, st = o.spikes()
    assert list(sc) == [0, 0, 0, 0] and np.array_equal(st, sched[:4])
    g = sum(0.0002 * np.exp(-(12.0 - (s + 1.25)) / 3.0) for s in sched[:4])
    assert o.syn_g()[0] == pytest.approx(g, rel=1e-13)
    assert o.voltage()[1] > -65.0


def test_k3_mixed_network_invariants(orc):
    """Sources, LIF and cable cells in one network: sources fire their schedule, LIF spikes coincide with event times
    (spike time - delay is a spike of a presynaptic cell), refractory gaps hold, results do not depend on threads."""
    m = W.mixed_network()
    o = orc.Oracle(m)
    o.advance(60.0, m["dt"])
    sc, st = o.spikes()
    kind = m["cell_kind"]
    for c in np.flatnonzero(kind == 2):
        a, b = m["src_off"][c], m["src_off"][c + 1]
        assert np.array_equal(np.sort(st[sc == c]), m["src_time"][a:b][m["src_time"][a:b] < 60.0])
    n_lif_spikes = 0
    for c in np.flatnonzero(kind == 1):
        mine = np.sort(st[sc == c])
        n_lif_spikes += len(mine)
        assert np.all(np.diff(mine) >= m["lif_t_ref"][c])
        pre = np.flatnonzero(m["conn_dst"] == c)
        arrivals = np.concatenate([st[sc == m["conn_src"][k]] + m["conn_delay"][k] for k in pre])
        for x in mine:
            assert np.min(np.abs(arrivals - x)) < 1e-12
    assert n_lif_spikes > 20 and np.count_nonzero(kind[sc] == 0) > 3
    o2 = orc.Oracle(m, threads=4)
    o2.advance(60.0, m["dt"])
    assert np.array_equal(o2.voltage(), o.voltage()) and np.array_equal(o2.spikes()[1], st)
