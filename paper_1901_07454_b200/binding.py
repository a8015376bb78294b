"""Thin Python binding of libarbb200.so (include/arbb200.h).  Argument marshalling only: every step
of the path runs in the library's CUDA kernels.  PyTorch supplies device memory (the workspace
tensor) and the stream; there is no CPU fallback - importing this module without the built library,
or creating a model without a CUDA device, raises.
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libarbb200.so")

ARB_OK, ARB_E_NULL, ARB_E_INVALID, ARB_E_WORKSPACE, ARB_E_CUDA, ARB_E_OVERFLOW, ARB_E_NOMEM, ARB_E_DIVERGED = 0, -1, -2, -3, -4, -5, -6, -7
ARB_PROBE_M, ARB_PROBE_H, ARB_PROBE_N, ARB_PROBE_SYN_G, ARB_PROBE_TIME, ARB_PROBE_NSTEPS, ARB_PROBE_STATS, ARB_PROBE_TIMING = range(8)
ARB_OPT_FUSED_STEPS, ARB_OPT_EPOCH_STEPS, ARB_OPT_TIMING, ARB_OPT_OVERLAP, ARB_OPT_L2_PREFETCH, ARB_OPT_GROUP_CTAS, ARB_OPT_HOT_FIRST = 1, 2, 3, 4, 5, 6, 7
ARB_OPT_LINEARISED = 8

EXPORTS = ("arb_plan", "arb_create", "arb_advance", "arb_spikes", "arb_clear_spikes", "arb_spike_block", "arb_apply_spike_blocks",
           "arb_voltage", "arb_probe", "arb_gates_noalloc", "arb_noalloc_max_cv", "arb_catalogue_size", "arb_catalogue_entry", "arb_catalogue_param", "arb_catalogue_find",
           "arb_set_state", "arb_set_option", "arb_fp64_peak", "arb_destroy", "arb_last_error")

# arb_desc's layout / capacity options (0 = library default).  A workloads dict may carry them under the
# same names; LAYOUT_DEFAULTS fills in the ones it does not (the parity tests run every case under
# several layouts this way).
OPTION_FIELDS = ("layout_group_min_cells", "layout_forest_cv", "cap_spikes", "cap_events", "shard_gid_base", "shard_n_global")
LAYOUT_DEFAULTS = {}


class ArbError(RuntimeError):
    def __init__(self, code, text):
        super().__init__("arbb200 error %d: %s" % (code, text))
        self.code = code


class arb_desc(C.Structure):
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
        ("layout_group_min_cells", C.c_int64), ("layout_forest_cv", C.c_int64),
        ("cap_spikes", C.c_int64), ("cap_events", C.c_int64),
        ("shard_gid_base", C.c_int64), ("shard_n_global", C.c_int64),
        ("cell_kind", C.c_void_p),
        ("lif_tau_m", C.c_void_p), ("lif_v_th", C.c_void_p), ("lif_c_m", C.c_void_p), ("lif_e_l", C.c_void_p),
        ("lif_e_r", C.c_void_p), ("lif_t_ref", C.c_void_p),
        ("src_off", C.c_void_p), ("src_time", C.c_void_p),
    ]


_lib = None


def lib():
    """The loaded library.  Fails loudly when it has not been built."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError("libarbb200.so is not built: run `python -m paper_1901_07454_b200.build` "
                              "(or __graft_entry__.build()); there is no fallback path")
        L = C.CDLL(LIB_PATH)
        L.arb_plan.argtypes = [C.c_void_p, C.POINTER(C.c_size_t)]
        L.arb_create.argtypes = [C.c_void_p, C.c_void_p, C.c_size_t, C.c_void_p, C.c_void_p]
        L.arb_advance.argtypes = [C.c_void_p, C.c_double, C.c_double]
        L.arb_spikes.restype = C.c_int64
        L.arb_spikes.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int64]
        L.arb_voltage.argtypes = [C.c_void_p, C.c_void_p, C.c_int64]
        L.arb_probe.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_int64]
        L.arb_gates_noalloc.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_int64]
        L.arb_noalloc_max_cv.restype = C.c_int64
        L.arb_noalloc_max_cv.argtypes = []
        L.arb_set_state.argtypes = [C.c_void_p] * 6
        L.arb_set_option.argtypes = [C.c_void_p, C.c_int, C.c_int64]
        L.arb_clear_spikes.argtypes = [C.c_void_p]
        L.arb_catalogue_entry.argtypes = [C.c_int, C.POINTER(C.c_char_p), C.POINTER(C.c_int), C.POINTER(C.c_int)]
        L.arb_catalogue_param.argtypes = [C.c_int, C.c_int, C.POINTER(C.c_char_p), C.POINTER(C.c_char_p), C.POINTER(C.c_double)]
        L.arb_catalogue_find.argtypes = [C.c_char_p]
        L.arb_spike_block.restype = C.c_int64
        L.arb_spike_block.argtypes = [C.c_void_p, C.c_void_p, C.c_int64]
        L.arb_apply_spike_blocks.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_int64, C.c_int64]
        L.arb_fp64_peak.argtypes = [C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.arb_destroy.argtypes = [C.c_void_p]
        L.arb_destroy.restype = None
        L.arb_last_error.restype = C.c_char_p
        L.arb_last_error.argtypes = [C.c_void_p]
        _lib = L
    return _lib


def _ptr(a):
    return None if a is None else a.ctypes.data


def make_desc(m):
    """arb_desc over the NumPy arrays of a workloads dict (the dict must outlive the call)."""
    d = arb_desc()
    for name, _ in arb_desc._fields_:
        v = m.get(name)
        if name in OPTION_FIELDS:
            setattr(d, name, int(v if v is not None else LAYOUT_DEFAULTS.get(name, 0)))
        elif isinstance(v, np.ndarray):
            setattr(d, name, _ptr(v))
        elif v is None:
            setattr(d, name, None)
        else:
            setattr(d, name, v)
    return d


def arb_fp64_peak(stream=None):
    """(DFMA per second, ms of the timed launch) of the current CUDA device; `stream` = a cudaStream_t handle."""
    r, ms = C.c_double(0.0), C.c_double(0.0)
    rc = lib().arb_fp64_peak(C.c_void_p(stream or 0), C.byref(r), C.byref(ms))
    if rc:
        raise ArbError(rc, "arb_fp64_peak failed")
    return r.value, ms.value


def catalogue():
    """The library's mechanism catalogue as {name: (kind, [(arb_desc field, unit, default), ...])}."""
    L, out = lib(), {}
    for i in range(L.arb_catalogue_size()):
        name, kind, n = C.c_char_p(), C.c_int(), C.c_int()
        L.arb_catalogue_entry(i, C.byref(name), C.byref(kind), C.byref(n))
        ps = []
        for j in range(n.value):
            f, u, d = C.c_char_p(), C.c_char_p(), C.c_double()
            L.arb_catalogue_param(i, j, C.byref(f), C.byref(u), C.byref(d))
            ps.append((f.value.decode(), u.value.decode(), d.value))
        out[name.value.decode()] = (kind.value, ps)
    return out


def arb_plan(m):
    d = make_desc(m)
    n = C.c_size_t(0)
    rc = lib().arb_plan(C.byref(d), C.byref(n))
    if rc:
        raise ArbError(rc, lib().arb_last_error(None).decode())
    return n.value


class Model:
    """arb_create / arb_advance / arb_spikes / arb_voltage / arb_probe on one CUDA device."""

    def __init__(self, m, device="cuda:0", stream=None):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("arbb200 needs a CUDA device; there is no CPU fallback")
        self._torch = torch
        self.n_cv, self.n_syn, self.n_cells = int(m["n_cv"]), int(m["n_syn"]), int(m["n_cells"])
        self.device = torch.device(device)
        self.workspace_bytes = arb_plan(m)
        with torch.cuda.device(self.device):
            self.workspace = torch.empty(self.workspace_bytes + 256, dtype=torch.uint8, device=self.device)
            self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
            base = self.workspace.data_ptr()
            aligned = (base + 255) // 256 * 256
            d = make_desc(m)
            self._h = C.c_void_p()
            rc = lib().arb_create(C.byref(d), C.c_void_p(aligned), C.c_size_t(self.workspace_bytes),
                                  C.c_void_p(self.stream.cuda_stream), C.byref(self._h))
        if rc:
            raise ArbError(rc, lib().arb_last_error(None).decode())

    def _check(self, rc):
        if rc < 0:
            raise ArbError(rc, lib().arb_last_error(self._h).decode())
        return rc

    def advance(self, t_end, dt):
        with self._torch.cuda.device(self.device):
            self._check(lib().arb_advance(self._h, float(t_end), float(dt)))

    def set_option(self, key, value):
        self._check(lib().arb_set_option(self._h, int(key), int(value)))

    def voltage(self, out=None):
        out = np.empty(self.n_cv) if out is None else out
        self._check(lib().arb_voltage(self._h, _ptr(out), self.n_cv))
        return out

    def probe(self, what):
        n = {ARB_PROBE_SYN_G: self.n_syn, ARB_PROBE_TIME: 1, ARB_PROBE_NSTEPS: 2, ARB_PROBE_STATS: 20,
             ARB_PROBE_TIMING: 4}.get(what, self.n_cv)
        out = np.empty(n)
        self._check(lib().arb_probe(self._h, what, _ptr(out), n))
        return out

    def gates(self):
        return self.probe(ARB_PROBE_M), self.probe(ARB_PROBE_H), self.probe(ARB_PROBE_N)

    def syn_g(self):
        return self.probe(ARB_PROBE_SYN_G)

    def gates_noalloc(self, what):
        """arb_gates_noalloc: one gate (ARB_PROBE_M / H / N) per CV through the library's static staging array."""
        out = np.empty(self.n_cv)
        self._check(lib().arb_gates_noalloc(self._h, int(what), _ptr(out), self.n_cv))
        return out

    def time(self):
        return float(self.probe(ARB_PROBE_TIME)[0])

    def stats(self):
        s = self.probe(ARB_PROBE_STATS)
        return dict(units=int(s[0]), slots=int(s[1]), branches=int(s[2]), workspace_bytes=int(s[3]),
                    events_delivered=int(s[4]), launches=int(s[5]), epoch_steps=int(s[6]),
                    streamed_bytes_per_step=int(s[7]), warp_units=int(s[8]), warps_per_cta=int(s[9]),
                    smem_per_warp=int(s[10]), topo_records=int(s[11]), groups=int(s[12]), classes=int(s[13]),
                    group_ctas=int(s[14]), group_smem=int(s[15]), forests=int(s[16]), block_units=int(s[17]),
                    forest_ctas=int(s[18]), forest_smem=int(s[19]))

    def timing(self):
        t = self.probe(ARB_PROBE_TIMING)
        return dict(cable_ms=float(t[0]), cable_launches=int(t[1]), event_ms=float(t[2]), event_launches=int(t[3]))

    def spikes(self):
        n = self._check(lib().arb_spikes(self._h, None, None, 0))
        cell, t = np.empty(n, np.int64), np.empty(n)
        if n:
            self._check(lib().arb_spikes(self._h, _ptr(cell), _ptr(t), n))
        return cell, t

    def spike_block(self, block, cap):
        """Fill `block` (a CUDA int64 tensor of 1 + 2 cap words) with the spikes since the last call; returns their count."""
        return self._check(lib().arb_spike_block(self._h, C.c_void_p(block.data_ptr()), int(cap)))

    def apply_spike_blocks(self, blocks, n_blocks, cap, own_block):
        self._check(lib().arb_apply_spike_blocks(self._h, C.c_void_p(blocks.data_ptr()), int(n_blocks), int(cap), int(own_block)))

    def clear_spikes(self):
        self._check(lib().arb_clear_spikes(self._h))

    def set_state(self, v=None, m=None, h=None, n=None, syn_g=None):
        arrs = [None if a is None else np.ascontiguousarray(a, np.float64) for a in (v, m, h, n, syn_g)]
        self._check(lib().arb_set_state(self._h, *[_ptr(a) for a in arrs]))

    def close(self):
        if getattr(self, "_h", None):
            lib().arb_destroy(self._h)
            self._h = C.c_void_p()
            self.workspace = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
