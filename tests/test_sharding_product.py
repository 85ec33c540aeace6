"""Product-path multi-rank test: world size 2, one process per rank, every rank compiles the
automaton on ITS device and decodes ITS contiguous row shard with cd_decode_loop (libcd.so, not the
oracle); rank 0 checks the rank-order concatenation against the oracle on the whole batch.

The path has no exchange step, so the ranks never wait for one another: with two devices each rank gets
its own; on a box with one device both ranks share cuda:0 (their kernels are independent launches that
time-slice the device -- nothing in them waits for the other process), so the rank logic, the per-rank
shard generation (`rows=` of workloads.build_step_logits) and the library under world_size > 1 are
exercised wherever at least one device is visible.  Result plumbing goes through gloo."""
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

pytestmark = pytest.mark.gpu


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _cfg():
    return wl.scaled(wl.CONFIGS["c3"], V=50000, B=1301, S=48, max_steps=9, density=0.03, accept_frac=0.2)


def _worker(rank: int, world: int, port: int, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        import paper_2606_31808_b200 as cd

        dev = f"cuda:{rank % torch.cuda.device_count()}"
        torch.cuda.set_device(dev)
        cfg = _cfg()
        aut = wl.build_automaton(cfg)
        lo, hi = wl.shard_rows(cfg.B, world, rank)
        # the rank's shard of the batch, byte-identical to those rows of the whole batch
        logits = wl.build_step_logits(cfg, aut, device=dev, rows=(lo, hi))
        dfa = cd.compile_dfa(aut.V, aut.S, aut.start, aut.row_ptr, aut.tok, aut.next, aut.accepting, device=dev)
        out = {}
        for name, mode in (("auto", cd.LOOP_AUTO), ("barrier", cd.LOOP_BARRIER), ("per_step", cd.LOOP_PER_STEP)):
            dfa.set_loop_mode(mode)
            res = cd.decode_loop(dfa, logits)
            out[name] = {k: v.cpu() for k, v in res.items()}
        before = cd.launch_count()
        assert before > 0
        dfa.close()
        payload = {"range": (lo, hi), "out": out, "lib": cd.lib_path()}
        gathered = [None] * world if rank == 0 else None
        dist.gather_object(payload, gathered, dst=0)
        if rank == 0:
            q.put(gathered)
        dist.barrier()
    finally:
        dist.destroy_process_group()


@pytest.mark.timeout(600)
def test_two_ranks_decode_their_shards_with_the_library(oracle):
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    world = 2
    ctx = mp.get_context("spawn")
    q = ctx.SimpleQueue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    gathered = q.get()
    for p in procs:
        p.join(120)
        assert p.exitcode == 0
    cfg = _cfg()
    aut = wl.build_automaton(cfg)
    # the whole batch, generated the same way on the device the shards came from (CPU and CUDA generators differ)
    full_logits = [x.cpu() for x in wl.build_step_logits(cfg, aut, device="cuda:0")]
    full = oracle.decode_loop(aut, full_logits)
    ranges = [g["range"] for g in gathered]
    assert ranges[0][0] == 0 and ranges[-1][1] == cfg.B and ranges[0][1] == ranges[1][0]
    for g in gathered:
        assert g["lib"].endswith("libcd.so")
    for mode in ("auto", "barrier", "per_step"):
        for key in ("tokens", "len", "final_state", "done"):
            cat = np.concatenate([g["out"][mode][key].numpy() for g in gathered], axis=0)
            assert np.array_equal(cat, full[key]), (mode, key)
        slp = np.concatenate([g["out"][mode]["sum_logprob"].numpy() for g in gathered]).astype(np.float64)
        assert np.all(np.abs(slp - full["sum_logprob"]) <= 1e-5 * (full["len"] + np.abs(full["sum_logprob"])) + 1e-12), mode
    assert int(full["n_active_hist"][0]) == cfg.B and int(full["n_active_hist"][-1]) < cfg.B
