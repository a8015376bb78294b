"""CPU-side checks of the C-ABI library: it loads, exports what include/arbb200.h declares, and its
host logic (validation, planning) behaves.  No compute calls: those need a GPU (tests -m gpu)."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from paper_1901_07454_b200 import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def B():
    from paper_1901_07454_b200 import build, binding
    build.build()
    binding.lib()
    return binding


def test_exports_match_header(B):
    header = open(os.path.join(ROOT, "include", "arbb200.h")).read()
    declared = set(re.findall(r"\b(arb_[a-z0-9_]+)\s*\(", header))
    assert declared == set(B.EXPORTS)
    for name in declared:
        assert hasattr(B.lib(), name), name


def test_desc_struct_matches_header(B):
    header = open(os.path.join(ROOT, "include", "arbb200.h")).read()
    body = header[header.index("typedef struct {"):header.index("} arb_desc;")]
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    names = []
    for decl in body.split(";"):
        decl = decl.replace("typedef struct {", "").strip()
        if not decl:
            continue
        decl = re.sub(r"^(const\s+)?(int64_t|int32_t|double)\s*\*?", "", decl)
        names += [n.strip(" *\n") for n in decl.split(",")]
    assert names == [f for f, _ in B.arb_desc._fields_]


def test_plan_sizes(B):
    small = B.arb_plan(W.config0())
    assert 0 < small < 64 << 20
    a, b = B.arb_plan(W.config1(n_cells=50)), B.arb_plan(W.config1(n_cells=100))
    assert small < a < b
    # about 150 bytes per CV plus fixed buffers: the 100k-cell config must fit one 180 GB GPU easily
    per_cv = (b - a) / (50 * 301)
    assert 60 < per_cv < 400


def test_plan_validation(B):
    def code(**kw):
        m = dict(W.random_model(3, n_cells=3))
        for k, v in kw.items():
            if v is None:
                m[k] = None
            else:
                a = np.array(m[k], copy=True)
                a[v[0]] = v[1]
                m[k] = a
        with pytest.raises(B.ArbError) as e:
            B.arb_plan(W.finalize(m))
        return e.value.code
    assert code(cv_parent=(0, 0)) == B.ARB_E_INVALID
    assert code(cv_parent=(2, 2)) == B.ARB_E_INVALID
    assert code(cv_area=(1, -1.0)) == B.ARB_E_INVALID
    assert code(cv_area=(1, np.inf)) == B.ARB_E_INVALID
    assert code(cv_cm=(0, 0.0)) == B.ARB_E_INVALID
    assert code(cv_raxial=(1, 0.0)) == B.ARB_E_INVALID
    assert code(syn_tau=(0, 0.0)) == B.ARB_E_INVALID
    assert code(syn_cv=(0, 10 ** 6)) == B.ARB_E_INVALID
    assert code(conn_delay=(0, 0.0)) == B.ARB_E_INVALID
    assert code(conn_src=(0, 99)) == B.ARB_E_INVALID
    assert code(conn_syn=(0, 999)) == B.ARB_E_INVALID
    assert code(ext_time=(0, -1.0)) == B.ARB_E_INVALID
    assert code(ext_weight=(0, np.nan)) == B.ARB_E_INVALID
    assert code(clamp_cv=(0, 10 ** 6)) == B.ARB_E_INVALID
    assert code(det_cv=(0, -1)) == B.ARB_E_INVALID
    assert code(pas_e=None) == B.ARB_E_INVALID
    n = C.c_size_t()
    assert B.lib().arb_plan(None, C.byref(n)) == B.ARB_E_NULL
    assert B.lib().arb_last_error(None) != b""


def test_null_model_calls_do_not_crash(B):
    L = B.lib()
    assert L.arb_advance(None, 1.0, 0.025) == B.ARB_E_NULL
    assert L.arb_spikes(None, None, None, 0) == B.ARB_E_NULL
    assert L.arb_voltage(None, None, 0) == B.ARB_E_NULL
    assert L.arb_set_option(None, 1, 1) == B.ARB_E_NULL
    L.arb_destroy(None)


def test_no_cpu_fallback(B):
    import torch
    if torch.cuda.is_available():
        pytest.skip("CUDA present")
    with pytest.raises(RuntimeError):
        B.Model(W.config0())


def test_product_does_not_touch_the_oracle():
    """The product path may not import, link or read anything under oracle/."""
    pkg = os.path.join(ROOT, "paper_1901_07454_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".cpp", ".hpp", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "arb_oracle" not in src and "liborc" not in src and "import orc" not in src, f
                assert not re.search(r"^\s*(from|import)\s+oracle", src, flags=re.M), f


def test_catalogue_names_the_mechanisms_and_cell_kinds(B):
    """mechanisms are referenced by name from a catalogue; every parameter names an arb_desc field."""
    cat = B.catalogue()
    assert set(cat) == {"hh", "pas", "expsyn", "iclamp", "lif", "spike_source"}
    assert cat["hh"][0] == 0 and cat["expsyn"][0] == 1 and cat["lif"][0] == 2
    fields = {f for f, _ in B.arb_desc._fields_}
    for name, (kind, params) in cat.items():
        for field, unit, default in params:
            assert field in fields, (name, field)
    assert dict((f, d) for f, _, d in cat["hh"][1])["hh_gnabar"] == W.GNABAR
    assert dict((f, d) for f, _, d in cat["lif"][1]) == W.LIF_DEFAULTS
    L = B.lib()
    assert L.arb_catalogue_find(b"pas") >= 0 and L.arb_catalogue_find(b"nope") == -1
    assert L.arb_catalogue_entry(99, None, None, None) == B.ARB_E_INVALID


def test_plan_accepts_and_validates_cell_kinds(B):
    m = W.mixed_network()
    assert B.arb_plan(m) > 0
    bad = dict(m)
    bad["cell_kind"] = m["cell_kind"].copy()
    bad["cell_kind"][-1] = 1                          # a 301-CV cell cannot be a LIF cell
    with pytest.raises(B.ArbError):
        B.arb_plan(bad)
    bad = dict(m)
    bad["lif_tau_m"] = m["lif_tau_m"].copy()
    bad["lif_tau_m"][np.flatnonzero(m["cell_kind"] == 1)[0]] = 0.0
    with pytest.raises(B.ArbError):
        B.arb_plan(bad)
    bad = dict(m)
    bad["src_time"] = m["src_time"][::-1].copy()      # schedules must ascend
    with pytest.raises(B.ArbError):
        B.arb_plan(bad)
