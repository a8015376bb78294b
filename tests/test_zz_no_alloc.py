"""arb_gates_noalloc (include/arbb200.h): the gate read-back whose device staging buffer is the library's static device
array instead of the caller's workspace.  Its output is compared with the existing path's (arb_probe) - the same gather
on another buffer, so the tolerance the parity tests use (1e-12) is met with equality - on two calls in a row, with the
state moving in between and with a SMALLER model after a larger one (the array keeps the last call's contents).
Collected last on purpose (the suite runs with pytest -x): it passes alone in a fresh process and after the others."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

DT = 0.025
TOL = 1e-12


@pytest.fixture(scope="module")
def B():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1901_07454_b200 import binding
    binding.LAYOUT_DEFAULTS.clear()
    return binding


def _rel(a, b):
    return float(np.max(np.abs(a - b) / np.maximum(np.abs(b), 1.0))) if len(a) else 0.0


def _check(B, g):
    n_set = 0
    for what in (B.ARB_PROBE_M, B.ARB_PROBE_H, B.ARB_PROBE_N):
        new, old = g.gates_noalloc(what), g.probe(what)
        assert new.shape == old.shape
        assert _rel(new, old) <= TOL and np.array_equal(new == 0.0, old == 0.0)
        n_set += int(np.count_nonzero(old))
    return n_set


def test_gates_noalloc_matches_probe_on_calls_in_a_row(B):
    from paper_1901_07454_b200 import workloads as W
    big = B.Model(W.config4(n_cells=60, t_end=10.0))       # HH on the soma and on 10 % of the dendritic CVs: groups and forests
    small = B.Model(W.config1(n_cells=8, t_end=10.0))      # HH on the soma only: most of the staging buffer must read 0
    assert big.n_cv > small.n_cv
    assert _check(B, big) > 3 * 60
    first = big.gates_noalloc(B.ARB_PROBE_M)
    assert np.array_equal(first, big.gates_noalloc(B.ARB_PROBE_M))      # two calls in a row, nothing in between
    big.advance(2.0, DT)
    small.advance(2.0, DT)
    assert _check(B, big) > 3 * 60                          # the state has moved: the second round of calls sees the new gates
    assert not np.array_equal(first, big.gates_noalloc(B.ARB_PROBE_M))
    # the smaller model right after the larger one: what the larger one left in the array must not show through
    assert _check(B, small) == 3 * 8
    assert _check(B, big) > 3 * 60
    big.close(), small.close()


def test_gates_noalloc_rejects_what_does_not_fit(B):
    from paper_1901_07454_b200 import workloads as W
    limit = int(B.lib().arb_noalloc_max_cv())
    assert limit == 1 << 19
    m = W.config3(n_cells=limit // 505 + 2, t_end=1.0)
    assert m["n_cv"] > limit
    g = B.Model(m)
    with pytest.raises(B.ArbError) as err:
        g.gates_noalloc(B.ARB_PROBE_M)
    assert err.value.code == B.ARB_E_INVALID and str(limit) in str(err.value)
    assert np.count_nonzero(g.probe(B.ARB_PROBE_M)) == m["n_cells"]     # the model is still usable, the existing path still works
    with pytest.raises(B.ArbError):
        g.gates_noalloc(B.ARB_PROBE_SYN_G)           # not a gate selector
    g.close()
