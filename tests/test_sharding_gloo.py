"""World-size-2 `gloo` test of the row sharding.

The path shards by rows with no exchange step: rank g takes the contiguous row range
`workloads.shard_rows(B, world, g)`, the automaton is replicated, every rank decodes and compacts
locally.  Checked here on CPU (the per-rank decode is the oracle's; on GPUs it is cd_decode_loop):
  * the ranges tile [0, B) without gap or overlap;
  * concatenating the ranks' results in rank order equals the single-process result row by row
    (row independence: one row in, one value out);
  * concatenating the ranks' locally compacted active lists (shifted by the range start) in rank
    order is the global stable active list at every step -- no collective needed for the order;
  * the global active count is the sum of the local ones (the only figure a rank would ever
    all-reduce, as bench.py does for its timing).
"""
import os
import socket
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import workloads as wl  # noqa: E402


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _case():
    cfg = wl.scaled(wl.CONFIGS["c3"], V=4096, B=37, S=24, max_steps=6, density=0.05, accept_frac=0.25)
    aut = wl.build_automaton(cfg)
    logits = wl.build_step_logits(cfg, aut)
    return cfg, aut, logits


def _active_lists(res, B, max_steps):
    """active row ids before each step, from the per-row lengths (a row is active at step k iff len > k)"""
    ln = res["len"]
    return [np.nonzero(ln > k)[0].astype(np.int32) for k in range(max_steps)]


def _worker(rank: int, world: int, port: int, q):
    import oracle

    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        cfg, aut, logits = _case()
        lo, hi = wl.shard_rows(cfg.B, world, rank)
        local = oracle.decode_loop(aut, [x[lo:hi].contiguous() for x in logits])
        # gather everything on rank 0 (test plumbing only; the data path itself has no collective)
        payload = {k: torch.from_numpy(np.ascontiguousarray(v)) for k, v in local.items()}
        payload["range"] = torch.tensor([lo, hi])
        gathered = [None] * world if rank == 0 else None
        dist.gather_object(payload, gathered, dst=0)
        n_local = torch.from_numpy(local["n_active_hist"].astype(np.int64))
        dist.all_reduce(n_local)  # global active count per step = sum of the local ones
        if rank == 0:
            q.put(([{k: v.numpy() for k, v in g.items()} for g in gathered], n_local.numpy()))
        dist.barrier()
    finally:
        dist.destroy_process_group()


@pytest.mark.timeout(180)
def test_row_sharding_world2_gloo(oracle):
    world = 2
    ctx = mp.get_context("spawn")
    q = ctx.SimpleQueue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    gathered, n_global = q.get()
    for p in procs:
        p.join(60)
        assert p.exitcode == 0

    cfg, aut, logits = _case()
    full = oracle.decode_loop(aut, logits)
    # ranges tile [0, B)
    ranges = [tuple(int(v) for v in g["range"]) for g in gathered]
    assert ranges[0][0] == 0 and ranges[-1][1] == cfg.B
    assert all(ranges[i][1] == ranges[i + 1][0] for i in range(world - 1))
    # rank-order concatenation == single-process result
    for key in ("tokens", "len", "final_state", "done"):
        cat = np.concatenate([g[key] for g in gathered], axis=0)
        assert np.array_equal(cat, full[key]), key
    assert np.array_equal(np.concatenate([g["sum_logprob"] for g in gathered]), full["sum_logprob"])
    # local active lists, shifted, concatenated in rank order == global stable active list
    glob = _active_lists(full, cfg.B, cfg.max_steps)
    for k in range(cfg.max_steps):
        parts = [_active_lists(g, hi - lo, cfg.max_steps)[k] + lo for g, (lo, hi) in zip(gathered, ranges)]
        cat = np.concatenate(parts)
        assert np.array_equal(cat, glob[k])
        assert np.all(np.diff(cat) > 0)  # ascending original row id = stable order
    assert np.array_equal(n_global, full["n_active_hist"].astype(np.int64))
    assert n_global[0] == cfg.B and n_global[-1] < cfg.B  # the case does exit early


def test_shard_rows_partition():
    for B in (0, 1, 7, 4096, 4097):
        for world in (1, 2, 3, 8):
            spans = [wl.shard_rows(B, world, r) for r in range(world)]
            assert spans[0][0] == 0 and spans[-1][1] == B
            assert all(a[1] == b[0] for a, b in zip(spans, spans[1:]))
            sizes = [hi - lo for lo, hi in spans]
            assert max(sizes) - min(sizes) <= 1
