"""ctypes binding of the CPU oracle (oracle/arb_oracle.c).

TEST INFRASTRUCTURE: only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
`--impl reference` legs may import this module.  It imports nothing from the product package and
shares no marshalling code with it; both sides read the same dict of NumPy arrays produced by
paper_1901_07454_b200.workloads (inputs only).
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = [os.path.join(_HERE, "arb_oracle.c"), os.path.join(_HERE, "arb_oracle.h")]
_LIB = os.path.join(_HERE, "liborc.so")
# tests/test_oracle_mutations.py points this at deliberately broken builds to show that the pins catch them
_LIB_OVERRIDE = os.environ.get("ORC_MUTANT_LIB")
CFLAGS = ["-O2", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-fPIC", "-shared", "-std=c11",
          "-Wall"]

PROBE_M, PROBE_H, PROBE_N, PROBE_SYN_G, PROBE_TIME, PROBE_NSTEPS = range(6)


def build(force=False):
    """Compile the oracle with gcc (plain C, no contraction).  Building the checker is not using it."""
    if not force and os.path.exists(_LIB) and all(os.path.getmtime(_LIB) >= os.path.getmtime(s) for s in _SRC):
        return _LIB
    subprocess.check_call(["gcc", *CFLAGS, "-o", _LIB, _SRC[0], "-lm"])
    return _LIB


class _Desc(C.Structure):
    _fields_ = [
        ("n_cells", C.c_int64), ("cv_off", C.c_void_p), ("cv_parent", C.c_void_p),
        ("cv_area", C.c_void_p), ("cv_cm", C.c_void_p), ("cv_raxial", C.c_void_p),
        ("cv_vinit", C.c_void_p),
        ("hh_gnabar", C.c_void_p), ("hh_gkbar", C.c_void_p), ("hh_gl", C.c_void_p),
        ("hh_ena", C.c_double), ("hh_ek", C.c_double), ("hh_el", C.c_double),
        ("pas_g", C.c_void_p), ("pas_e", C.c_void_p),
        ("syn_off", C.c_void_p), ("syn_cv", C.c_void_p), ("syn_tau", C.c_void_p), ("syn_e", C.c_void_p),
        ("n_clamp", C.c_int64), ("clamp_cell", C.c_void_p), ("clamp_cv", C.c_void_p),
        ("clamp_t0", C.c_void_p), ("clamp_t1", C.c_void_p), ("clamp_amp", C.c_void_p),
        ("det_cv", C.c_void_p), ("threshold", C.c_double),
        ("n_conn", C.c_int64), ("conn_src", C.c_void_p), ("conn_dst", C.c_void_p),
        ("conn_syn", C.c_void_p), ("conn_delay", C.c_void_p), ("conn_weight", C.c_void_p),
        ("n_ext", C.c_int64), ("ext_cell", C.c_void_p), ("ext_syn", C.c_void_p),
        ("ext_time", C.c_void_p), ("ext_weight", C.c_void_p),
        ("cell_kind", C.c_void_p),
        ("lif_tau_m", C.c_void_p), ("lif_v_th", C.c_void_p), ("lif_c_m", C.c_void_p), ("lif_e_l", C.c_void_p),
        ("lif_e_r", C.c_void_p), ("lif_t_ref", C.c_void_p),
        ("src_off", C.c_void_p), ("src_time", C.c_void_p),
    ]


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_LIB_OVERRIDE or build())
        L.orc_exprelr.restype = C.c_double
        L.orc_exprelr.argtypes = [C.c_double]
        L.orc_hh_rates.argtypes = [C.c_double, C.c_void_p]
        L.orc_assemble.argtypes = [C.c_int64] + [C.c_void_p] * 6 + [C.c_double] + [C.c_void_p] * 3
        L.orc_hines_solve.argtypes = [C.c_int64] + [C.c_void_p] * 5
        L.orc_create.argtypes = [C.c_void_p, C.c_void_p]
        L.orc_advance.argtypes = [C.c_void_p, C.c_double, C.c_double]
        L.orc_spikes.restype = C.c_int64
        L.orc_spikes.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int64]
        L.orc_voltage.argtypes = [C.c_void_p, C.c_void_p, C.c_int64]
        L.orc_probe.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_int64]
        L.orc_cell_currents.argtypes = [C.c_void_p, C.c_int64, C.c_void_p]
        L.orc_set_state.argtypes = [C.c_void_p] * 6
        L.orc_set_linearised.argtypes = [C.c_void_p, C.c_int]
        L.orc_set_threads.argtypes = [C.c_int]
        L.orc_get_threads.restype = C.c_int
        L.orc_destroy.argtypes = [C.c_void_p]
        L.orc_last_error.restype = C.c_char_p
        _lib = L
    return _lib


def _p(a):
    return None if a is None else a.ctypes.data


class OracleError(RuntimeError):
    pass


def exprelr(x):
    return lib().orc_exprelr(float(x))


def hh_rates(v):
    out = np.empty(6)
    lib().orc_hh_rates(float(v), _p(out))
    return out


def assemble(parent, area, cm, raxial, v, i_memb, delta):
    n = len(parent)
    parent = np.ascontiguousarray(parent, np.int32)
    arrs = [np.ascontiguousarray(a, np.float64) for a in (area, cm, raxial, v, i_memb)]
    d, u, rhs = np.empty(n), np.empty(n), np.empty(n)
    lib().orc_assemble(n, _p(parent), *[_p(a) for a in arrs], float(delta), _p(d), _p(u), _p(rhs))
    return d, u, rhs


def hines_solve(parent, d, u, rhs):
    n = len(parent)
    parent = np.ascontiguousarray(parent, np.int32)
    d, rhs = np.array(d, np.float64), np.array(rhs, np.float64)
    u = np.ascontiguousarray(u, np.float64)
    x = np.empty(n)
    lib().orc_hines_solve(n, _p(parent), _p(d), _p(u), _p(rhs), _p(x))
    return x


class Oracle:
    """The reference simulation: create from a workloads dict, advance, read back."""

    def __init__(self, m, threads=1):
        self._keep = m
        d = _Desc()
        for name, _ in _Desc._fields_:
            v = m.get(name)
            if isinstance(v, np.ndarray):
                setattr(d, name, _p(v))
            elif v is None:
                setattr(d, name, None)
            else:
                setattr(d, name, v)
        self.n_cv, self.n_syn, self.n_cells = m["n_cv"], m["n_syn"], m["n_cells"]
        self._h = C.c_void_p()
        lib().orc_set_threads(int(threads))
        self._check(lib().orc_create(C.byref(d), C.byref(self._h)))

    def _check(self, rc):
        if rc < 0:
            raise OracleError("oracle error %d: %s" % (rc, lib().orc_last_error().decode()))

    def advance(self, t_end, dt):
        self._check(lib().orc_advance(self._h, float(t_end), float(dt)))

    def voltage(self):
        out = np.empty(self.n_cv)
        self._check(lib().orc_voltage(self._h, _p(out), self.n_cv))
        return out

    def probe(self, what):
        n = {PROBE_SYN_G: self.n_syn, PROBE_TIME: 1, PROBE_NSTEPS: 2}.get(what, self.n_cv)
        out = np.empty(n)
        self._check(lib().orc_probe(self._h, what, _p(out), n))
        return out

    def gates(self):
        return self.probe(PROBE_M), self.probe(PROBE_H), self.probe(PROBE_N)

    def syn_g(self):
        return self.probe(PROBE_SYN_G)

    def time(self):
        return float(self.probe(PROBE_TIME)[0])

    def spikes(self):
        n = lib().orc_spikes(self._h, None, None, 0)
        cell, t = np.empty(n, np.int64), np.empty(n)
        if n:
            lib().orc_spikes(self._h, _p(cell), _p(t), n)
        return cell, t

    def currents(self, cell):
        off = self._keep["cv_off"]
        out = np.empty(int(off[cell + 1] - off[cell]))
        self._check(lib().orc_cell_currents(self._h, int(cell), _p(out)))
        return out

    def set_state(self, v=None, m=None, h=None, n=None, syn_g=None):
        arrs = [None if a is None else np.ascontiguousarray(a, np.float64) for a in (v, m, h, n, syn_g)]
        self._check(lib().orc_set_state(self._h, *[_p(a) for a in arrs]))

    def set_linearised(self, on=True):
        self._check(lib().orc_set_linearised(self._h, 1 if on else 0))

    def close(self):
        if self._h:
            lib().orc_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
