"""One network over several GPUs: cells are split into
contiguous ranges balanced by control-volume count, every rank holds the connections whose DESTINATION it owns
(sources stay global ids), and once per minimum-delay epoch the ranks all-gather fixed-capacity spike blocks and
push the other ranks' spikes through their own connection tables.

Host logic only - partitioning, marshalling, the epoch loop.  The integration and the spike -> event walk run in
the library's kernels (arb_advance, arb_spike_block, arb_apply_spike_blocks); the all-gather is
torch.distributed's (NCCL over NVLink on a multi-GPU box; the spike blocks are a few KB, so one fused gather per
epoch is latency-bound by design).  `LocalGroup` runs the ranks of one process one after the other on a single
GPU - the same calls in the same order - which is how the path is tested where only one GPU is available.

overlap=True (the exchange is hidden behind the integration of the next interval): the exchange epoch
is HALF the minimum delay, and the all-gather of the spikes of half-epoch h runs on NCCL's stream while half-epoch h + 1
is integrated; its spikes are applied before half-epoch h + 2, which is early enough because a spike of half-epoch h
cannot cause an event before its end plus half a minimum delay.  Results do not depend on the mode beyond rounding
(events are applied in (time, synapse, weight) order whenever they were queued).
"""
from __future__ import annotations

import numpy as np

_PER_CV = ("cv_parent", "cv_area", "cv_cm", "cv_raxial", "cv_vinit", "hh_gnabar", "hh_gkbar", "hh_gl", "pas_g", "pas_e")
_PER_SYN = ("syn_cv", "syn_tau", "syn_e")


def partition(cv_off, n_ranks):
    """Contiguous cell ranges [lo, hi) per rank, balanced by control-volume count."""
    cv_off = np.asarray(cv_off, np.int64)
    n_cells, total = len(cv_off) - 1, int(cv_off[-1])
    bounds = [0]
    for r in range(1, n_ranks):
        # first cell whose start lies at or beyond the r-th share of the control volumes
        cut = int(np.searchsorted(cv_off, total * r / n_ranks, side="left"))
        bounds.append(min(max(cut, bounds[-1]), n_cells))
    bounds.append(n_cells)
    return [(bounds[r], bounds[r + 1]) for r in range(n_ranks)]


def shard(m, lo, hi):
    """The part of network `m` (a workloads dict) that the owner of cells [lo, hi) needs: its cells, the
    connections INTO them (conn_src global, conn_dst local), their external events and clamps."""
    n_cells = int(m["n_cells"])
    assert 0 <= lo <= hi <= n_cells
    off, so = m["cv_off"], m["syn_off"]
    a, b = int(off[lo]), int(off[hi])
    sa, sb = int(so[lo]), int(so[hi])
    out = dict(n_cells=hi - lo, cv_off=off[lo:hi + 1] - a, syn_off=so[lo:hi + 1] - sa,
               n_cv=b - a, n_syn=sb - sa, shard_gid_base=lo, shard_n_global=n_cells)
    for k in ("t_end", "dt", "threshold", "hh_ena", "hh_ek", "hh_el"):
        if k in m:
            out[k] = m[k]
    for k in _PER_CV:
        out[k] = None if m.get(k) is None else np.ascontiguousarray(m[k][a:b])
    for k in _PER_SYN:
        out[k] = np.ascontiguousarray(m[k][sa:sb])
    out["det_cv"] = None if m.get("det_cv") is None else np.ascontiguousarray(m["det_cv"][lo:hi])
    sel = np.flatnonzero((m["conn_dst"] >= lo) & (m["conn_dst"] < hi))
    out["conn_src"] = np.ascontiguousarray(m["conn_src"][sel])
    out["conn_dst"] = np.ascontiguousarray(m["conn_dst"][sel] - lo)
    for k in ("conn_syn", "conn_delay", "conn_weight"):
        out[k] = np.ascontiguousarray(m[k][sel])
    sel = np.flatnonzero((m["ext_cell"] >= lo) & (m["ext_cell"] < hi))
    out["ext_cell"] = np.ascontiguousarray(m["ext_cell"][sel] - lo)
    for k in ("ext_syn", "ext_time", "ext_weight"):
        out[k] = np.ascontiguousarray(m[k][sel])
    sel = np.flatnonzero((m["clamp_cell"] >= lo) & (m["clamp_cell"] < hi))
    out["clamp_cell"] = np.ascontiguousarray(m["clamp_cell"][sel] - lo)
    for k in ("clamp_cv", "clamp_t0", "clamp_t1", "clamp_amp"):
        out[k] = np.ascontiguousarray(m[k][sel])
    out["n_conn"], out["n_ext"], out["n_clamp"] = len(out["conn_src"]), len(out["ext_cell"]), len(out["clamp_cell"])
    for k in ("layout_group_min_cells", "layout_forest_cv", "cap_spikes", "cap_events"):
        if k in m:
            out[k] = m[k]
    return out


def epoch_steps(min_delay, dt):
    """Grid steps of one exchange epoch: the library's rule (include/arbb200.h, arb_advance) on the GLOBAL minimum delay."""
    return max(1, min(1024, int(np.floor(min_delay / dt - 1e-6))))


def exchange_steps(min_delay, dt, overlap):
    """Grid steps between exchanges.  overlap: half an epoch, so that the spikes of one half-epoch may arrive while the
    next is integrated (None when the epoch is a single grid step: nothing to hide the exchange behind)."""
    if not np.isfinite(min_delay):
        return 1024
    es = epoch_steps(min_delay, dt)
    if not overlap:
        return es
    return es // 2 if es >= 2 else None


def exchange_point(t0, j, es, dt, t_end):
    """The j-th exchange point of a call that started at t0 (by multiplication, like the library's grid), or t_end when
    that is nearer than a rounding error (no sliver of a step at the end of a call)."""
    t = t0 + (j * es) * dt
    return t_end if t_end - t < 1e-9 * dt else t


def block_words(cap):
    return 1 + 2 * int(cap)


class DistGroup:
    """The exchange over torch.distributed (NCCL on GPUs): one all_gather_into_tensor of the spike blocks per epoch."""

    def __init__(self, torch, device):
        import torch.distributed as dist
        self.torch, self.dist, self.device = torch, dist, device
        self.rank, self.size = dist.get_rank(), dist.get_world_size()

    def min_delay(self, local_min):
        t = self.torch.tensor([float(local_min)], dtype=self.torch.float64, device=self.device)
        self.dist.all_reduce(t, op=self.dist.ReduceOp.MIN)
        return float(t.item())

    def all_gather(self, block, out, async_op=False):
        """Returns None, or (async_op) a handle whose wait() orders the gather before later work of the current stream."""
        return self.dist.all_gather_into_tensor(out, block, async_op=async_op)


class ShardedModel:
    """One rank's part of a sharded network: arb_create on its shard, and the epoch loop with the exchange."""

    def __init__(self, binding, m_global, rank, n_ranks, group, device="cuda:0", block_cap=None, ranges=None, local=None,
                 overlap=False):
        """m_global: the whole network (every rank cuts its shard out of it), or None with `local` = this rank's shard
        generated on its own (a workloads dict with shard_gid_base / shard_n_global set)."""
        import torch
        self.B, self.torch, self.rank, self.n_ranks, self.group = binding, torch, rank, n_ranks, group
        if local is None:
            self.ranges = ranges or partition(m_global["cv_off"], n_ranks)
            lo, hi = self.ranges[rank]
            self.local = shard(m_global, lo, hi)
        else:
            self.local = local
            lo = int(local["shard_gid_base"])
            hi = lo + int(local["n_cells"])
            self.ranges = ranges
        self.model = binding.Model(self.local, device=device)
        self.cap = int(block_cap or max(1024, 4 * (hi - lo)))
        self.overlap = bool(overlap)
        # two of each: with overlap, the blocks of one half-epoch are in flight while the next one is written
        self.block2 = [torch.zeros(block_words(self.cap), dtype=torch.int64, device=device) for _ in range(2)]
        self.blocks2 = [torch.zeros(n_ranks * block_words(self.cap), dtype=torch.int64, device=device) for _ in range(2)]
        self.block, self.blocks = self.block2[0], self.blocks2[0]
        local_min = float(np.min(self.local["conn_delay"])) if self.local["n_conn"] else float("inf")
        self.min_delay = group.min_delay(local_min) if group is not None else local_min
        self.t = 0.0

    def advance(self, t_end, dt):
        """Integrate to t_end in exchange epochs of floor(min_delay / dt) grid steps; spikes are exchanged after each.
        overlap: epochs of half that length, the exchange of one hidden behind the integration of the next."""
        es = exchange_steps(self.min_delay, dt, self.overlap)
        t0 = self.t                        # exchange points of this call: t0 + j es dt (by multiplication, like the library's grid)
        if not self.overlap or es is None:
            es = es or epoch_steps(self.min_delay, dt)
            j = 0
            while self.t < t_end:
                j += 1
                self.t = exchange_point(t0, j, es, dt, t_end)
                self.model.advance(self.t, dt)
                self.exchange()
            return
        pending, h = None, 0               # (work handle, blocks buffer) of the half-epoch before the one being integrated
        while self.t < t_end:
            self.t = exchange_point(t0, h + 1, es, dt, t_end)
            self.model.advance(self.t, dt)
            if pending is not None:
                self._finish(pending)
            block, blocks = self.block2[h & 1], self.blocks2[h & 1]
            self.model.spike_block(block, self.cap)
            pending = None
            if self.group is not None and self.n_ranks > 1:
                pending = (self.group.all_gather(block, blocks, async_op=True), blocks)
            h += 1
        if pending is not None:
            self._finish(pending)          # a call ends with every exchange applied

    def _finish(self, pending):
        work, blocks = pending
        if work is not None:
            work.wait()
        self.model.apply_spike_blocks(blocks, self.n_ranks, self.cap, self.rank)

    def exchange(self):
        self.model.spike_block(self.block, self.cap)
        if self.group is not None and self.n_ranks > 1:
            self.group.all_gather(self.block, self.blocks)
            self.model.apply_spike_blocks(self.blocks, self.n_ranks, self.cap, self.rank)

    def close(self):
        self.model.close()


class LocalGroup:
    """All ranks in one process on one GPU, one after the other: the calls a multi-GPU run makes, in the same order,
    with the all-gather replaced by a copy.  For tests and for checking a partition on a single-GPU box."""

    def __init__(self, binding, m_global, n_ranks, device="cuda:0", block_cap=None, overlap=False):
        import torch
        self.torch, self.n_ranks, self.overlap = torch, n_ranks, bool(overlap)
        self.ranges = partition(m_global["cv_off"], n_ranks)
        self.ranks = [ShardedModel(binding, m_global, r, n_ranks, None, device, block_cap, self.ranges) for r in range(n_ranks)]
        self.min_delay = min(s.min_delay for s in self.ranks)
        for s in self.ranks:
            s.min_delay = self.min_delay
        self.cap = max(s.cap for s in self.ranks)
        for s in self.ranks:
            if s.cap != self.cap:
                s.cap = self.cap
                s.block = torch.zeros(block_words(self.cap), dtype=torch.int64, device=device)
        self.blocks = torch.zeros(n_ranks * block_words(self.cap), dtype=torch.int64, device=device)
        self.t = 0.0

    def advance(self, t_end, dt):
        es = exchange_steps(self.min_delay, dt, self.overlap)
        late = self.overlap and es is not None      # apply the blocks of half-epoch h after half-epoch h + 1, as the overlap does
        if es is None:
            es = epoch_steps(self.min_delay, dt)
        w = block_words(self.cap)
        pending, t0, j = None, self.t, 0
        while self.t < t_end:
            j += 1
            nxt = exchange_point(t0, j, es, dt, t_end)
            for s in self.ranks:
                s.model.advance(nxt, dt)
            if pending is not None:
                self._apply(pending)
            blocks = self.torch.zeros_like(self.blocks) if late else self.blocks
            for r, s in enumerate(self.ranks):
                s.model.spike_block(s.block, self.cap)
                blocks[r * w:(r + 1) * w].copy_(s.block)
            self.torch.cuda.synchronize()
            pending = blocks
            if not late:
                self._apply(pending)
                pending = None
            self.t = nxt
        if pending is not None:
            self._apply(pending)

    def _apply(self, blocks):
        for r, s in enumerate(self.ranks):
            s.model.apply_spike_blocks(blocks, self.n_ranks, self.cap, r)

    def gather(self, what):
        """Concatenate a per-CV / per-synapse read-back of all ranks in global order."""
        return np.concatenate([what(s.model) for s in self.ranks])

    def spikes(self):
        cs, ts = [], []
        for (lo, _), s in zip(self.ranges, self.ranks):
            c, t = s.model.spikes()
            cs.append(c + lo), ts.append(t)
        c, t = np.concatenate(cs), np.concatenate(ts)
        order = np.lexsort((c, t))
        return c[order], t[order]

    def close(self):
        for s in self.ranks:
            s.close()


# ------------------------------------------------------------------------------------------------
# CPU self-test of the host logic under torch.distributed (gloo, world_size >= 2): partition, shards, and the
# all-gather of spike blocks with a stand-in for the device calls (there is no CPU integration path).
# ------------------------------------------------------------------------------------------------
def _selftest():
    import json
    import os
    import torch
    import torch.distributed as dist
    from . import workloads as W
    dist.init_process_group("gloo")
    rank, world = dist.get_rank(), dist.get_world_size()
    m = W.config3(n_cells=40, t_end=10.0)
    ranges = partition(m["cv_off"], world)
    lo, hi = ranges[rank]
    local = shard(m, lo, hi)
    group = DistGroup(torch, torch.device("cpu"))
    gmin = group.min_delay(float(np.min(local["conn_delay"])) if local["n_conn"] else float("inf"))
    cap = 64
    w = block_words(cap)
    ok = abs(gmin - float(np.min(m["conn_delay"]))) < 1e-15
    seen = []
    for epoch in range(3):
        # stand-in for arb_spike_block: every third local cell "fires" at a time that encodes (epoch, gid)
        gids = np.arange(lo, hi, dtype=np.int64)[(np.arange(lo, hi) + epoch) % 3 == 0]
        block = torch.zeros(w, dtype=torch.int64)
        block[0] = len(gids)
        block[1:1 + len(gids)] = torch.from_numpy(gids)
        block[1 + cap:1 + cap + len(gids)] = torch.from_numpy((epoch * 5.0 + gids * 1e-3).view(np.int64))
        blocks = torch.zeros(world * w, dtype=torch.int64)
        work = group.all_gather(block, blocks, async_op=(epoch == 1))      # the overlapped exchange uses the asynchronous form
        if work is not None:
            work.wait()
        got = []
        for r in range(world):
            n = int(blocks[r * w])
            got += list(zip(blocks[r * w + 1:r * w + 1 + n].tolist(),
                            blocks[r * w + 1 + cap:r * w + 1 + cap + n].numpy().view(np.float64).tolist()))
        want = [(int(g), epoch * 5.0 + g * 1e-3) for g in range(m["n_cells"]) if (g + epoch) % 3 == 0]
        ok = ok and sorted(got) == sorted(want)
        seen.append(len(got))
    # every connection of the network is held by exactly one rank, with its global source id
    mine = torch.tensor([local["n_conn"]], dtype=torch.int64)
    dist.all_reduce(mine)
    ok = ok and int(mine.item()) == m["n_conn"] and bool(np.all(local["conn_src"] < m["n_cells"]))
    flag = torch.tensor([1 if ok else 0], dtype=torch.int64)
    dist.all_reduce(flag, op=dist.ReduceOp.MIN)
    if rank == 0:
        print(json.dumps({"selftest": "sharded", "world": world, "ok": bool(flag.item()), "spikes_per_epoch": seen,
                          "ranges": ranges, "min_delay": gmin}), flush=True)
    dist.destroy_process_group()


if __name__ == "__main__":
    _selftest()
