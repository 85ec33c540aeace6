"""BASELINE.json configs[4] at full size, EVERY row against the oracle ("batches 0, 127, 255; all
steps").  A module of its own: the three gather modes and the three loop modes all run on one set of
logits against one oracle pass per batch."""
import numpy as np
import pytest
import torch

import workloads as wl
import test_gpu_parity as tp
from test_gpu_parity import TOL, cd  # noqa: F401  (cd: the module-scoped fixture)

pytestmark = pytest.mark.gpu

C4_BATCHES = (0, 127, 255)  # "batches 0, 127, 255; all steps"


@pytest.mark.parametrize("batch", C4_BATCHES)
def test_loop_c4_every_row_of_three_batches(cd, oracle, batch):
    """BASELINE.json configs[4]: full batches (B = 4096, S = 4096, 16 steps, 32 GiB of logits each) in
    the launch configuration bench.py times, EVERY row compared with the oracle: tokens, len,
    final_state and done bit for bit, sum_logprob within 1e-5 * (len + |sum|).  The oracle is fed row
    chunks of 512 rows x 16 steps (4 GiB of host memory at a time; rows are independent, PAPER.md
    L106).  The three gather modes and the three loop modes all run on the same logits against one
    oracle pass."""
    cfg = wl.CONFIGS["c4"]
    free, _ = torch.cuda.mem_get_info()
    if free < 40 * 2**30:
        pytest.skip("needs ~34 GiB of device memory")
    aut = wl.build_automaton(cfg, device="cuda:0")
    logits = wl.build_step_logits(cfg, aut, device="cuda:0", batch=batch)
    # the oracle, chunk by chunk
    ref = dict(tokens=[], len=[], final_state=[], done=[], sum_logprob=[])
    for r0 in range(0, cfg.B, 512):
        sub = [x[r0:r0 + 512].cpu() for x in logits]
        part = oracle.decode_loop(aut, sub, max_steps=cfg.max_steps)
        for k in ref:
            ref[k].append(part[k])
        del sub
    ref = {k: np.concatenate(v) for k, v in ref.items()}
    assert int(ref["len"].sum()) > 8 * cfg.B  # ~11 row-steps per row
    for mode in ("dense", "gather_all", "gather_mixed"):
        tp._MODE["name"] = mode
        dfa = tp.dev_dfa(cd, aut)
        for lm in (cd.LOOP_AUTO, cd.LOOP_BARRIER, cd.LOOP_PER_STEP):
            dfa.set_loop_mode(lm)
            out = cd.decode_loop(dfa, logits, max_steps=cfg.max_steps)
            for k in ("tokens", "len", "final_state", "done"):
                assert np.array_equal(out[k].cpu().numpy(), ref[k]), (mode, lm, k)
            slp = out["sum_logprob"].cpu().numpy().astype(np.float64)
            bound = TOL * (ref["len"] + np.abs(ref["sum_logprob"]))
            assert np.all(np.abs(slp - ref["sum_logprob"]) <= bound), (mode, lm)
        dfa.close()
    tp._MODE["name"] = "dense"
    # properties that hold at any size (a second, independent look at the same outputs)
    toks, ln, fs, dn = ref["tokens"], ref["len"], ref["final_state"], ref["done"]
    acc = aut.accepting.numpy()
    assert np.array_equal(dn, acc[fs]) and bool(np.all((ln == cfg.max_steps) | (dn == 1)))
    assert bool(np.all((toks >= 0) == (np.arange(cfg.max_steps)[None, :] < ln[:, None])))


