"""Host logic of the sharded (multi-GPU) path, on CPU: the partition, the shards (validated by arb_plan, which needs
no GPU), and the per-epoch all-gather of spike blocks under torch.distributed with the gloo backend (world size 2)."""
import json
import os
import subprocess
import sys

import numpy as np
import pytest

from paper_1901_07454_b200 import sharded as S, workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_partition_is_contiguous_and_balanced_by_control_volumes():
    m = W.config4(n_cells=400, t_end=1.0)
    for n in (1, 2, 3, 8):
        r = S.partition(m["cv_off"], n)
        assert r[0][0] == 0 and r[-1][1] == 400 and all(a[1] == b[0] for a, b in zip(r, r[1:]))
        cv = np.array([m["cv_off"][hi] - m["cv_off"][lo] for lo, hi in r])
        biggest = int(np.max(np.diff(m["cv_off"])))
        assert cv.max() - cv.min() <= 2 * biggest          # within one (largest) cell of each other
    # more ranks than cells: empty ranges at the end, nothing lost
    r = S.partition(W.config0()["cv_off"], 3)
    assert sum(hi - lo for lo, hi in r) == 1


def test_shards_hold_every_connection_once_with_global_sources():
    from paper_1901_07454_b200 import build, binding as B
    build.build()
    m = W.config2(n_cells=60, t_end=20.0)
    ranges = S.partition(m["cv_off"], 3)
    seen = []
    for lo, hi in ranges:
        s = S.shard(m, lo, hi)
        assert s["shard_gid_base"] == lo and s["shard_n_global"] == 60
        assert np.all((s["conn_dst"] >= 0) & (s["conn_dst"] < hi - lo)) and np.all((s["conn_src"] >= 0) & (s["conn_src"] < 60))
        seen += list(zip(s["conn_src"].tolist(), (s["conn_dst"] + lo).tolist(), s["conn_syn"].tolist(), s["conn_delay"].tolist()))
        assert len(s["ext_cell"]) == int(np.count_nonzero((m["ext_cell"] >= lo) & (m["ext_cell"] < hi)))
        assert B.arb_plan(s) > 0                           # the library accepts the shard (host validation, no GPU)
    want = list(zip(m["conn_src"].tolist(), m["conn_dst"].tolist(), m["conn_syn"].tolist(), m["conn_delay"].tolist()))
    assert sorted(seen) == sorted(want)
    # a source id beyond the network is rejected
    s = S.shard(m, *ranges[0])
    s["conn_src"] = s["conn_src"].copy()
    s["conn_src"][0] = 60
    with pytest.raises(B.ArbError):
        B.arb_plan(s)


def test_two_rank_exchange_over_gloo():
    """world_size 2, gloo: global minimum delay by all-reduce, one all_gather_into_tensor of spike blocks per epoch,
    every rank ends up with every spike of the network; every connection is owned by exactly one rank."""
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", "29741", "-m", "paper_1901_07454_b200.sharded"]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=300, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    line = [l for l in r.stdout.splitlines() if l.startswith("{")][-1]
    j = json.loads(line)
    assert j["ok"] and j["world"] == 2 and j["ranges"][0][1] == j["ranges"][1][0]


def test_exchange_steps_with_and_without_overlap():
    """Exchange epochs: the library's epoch rule on the global minimum delay; half of it when the exchange is hidden
    behind the next half-epoch's integration; no overlap when the epoch is a single grid step."""
    from paper_1901_07454_b200 import sharded as S
    assert S.exchange_steps(5.0, 0.025, False) == S.epoch_steps(5.0, 0.025) == 199      # the 1e-6 guard (R11/R12)
    assert S.exchange_steps(5.0, 0.025, True) == 99
    assert S.exchange_steps(7.3, 0.025, True) == 145 and 2 * 145 * 0.025 <= 7.3      # floor(291 / 2)
    assert S.exchange_steps(0.03, 0.025, True) is None
    assert S.exchange_steps(float("inf"), 0.025, True) == 1024
    assert S.exchange_point(0.0, 2, 100, 0.025, 5.0) == 5.0 and S.exchange_point(0.0, 1, 100, 0.025, 5.0) == 2.5
