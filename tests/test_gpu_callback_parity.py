"""Callback forms of the loops (cd_decode_loop_cb / cd_head_decode_loop_cb; "how a real LM
forward would plug in"): the callback is handed the device-side active list and returns the step's
logits / hidden states, indexed by original row id or as a compact batch (row = active slot) gathered on
the device without any host synchronisation.  Results must equal the oracle's loop bit for bit."""
import numpy as np
import pytest
import torch

import workloads as wl

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def cd():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    import paper_2606_31808_b200 as m

    m.lib()
    return m


@pytest.mark.parametrize("by_slot", [False, True])
@pytest.mark.parametrize("gather", [0, -1])
def test_logits_callback_loop(cd, oracle, by_slot, gather):
    V, B, steps = 3000, 300, 8
    aut = wl.make_random_dfa(61, V, 20, 0.1, 0.15)
    dfa = cd.compile_dfa(aut.V, aut.S, aut.start, aut.row_ptr, aut.tok, aut.next, aut.accepting, device="cuda:0")
    dfa.set_gather_max(gather)
    logits = [wl.make_logits(61, k, B, V, 2.0, torch.bfloat16) for k in range(steps)]
    dev = [x.to("cuda:0") for x in logits]
    calls = []

    def next_logits(step, row_ids, n_active):
        calls.append(step)
        if not by_slot:
            return dev[step], False
        # a "forward over the active rows": compact batch, gathered on the device, no host sync;
        # slots beyond n_active hold stale ids -> clamp, their rows are never read
        return dev[step].index_select(0, row_ids.long().clamp_(0, B - 1)), True

    got = cd.decode_loop_cb(dfa, next_logits, torch.bfloat16, B, steps)
    torch.cuda.synchronize()
    want = oracle.decode_loop(aut, logits)
    assert calls == list(range(steps))
    for k in ("tokens", "len", "final_state", "done"):
        assert np.array_equal(got[k].cpu().numpy(), want[k]), k
    err = np.abs(got["sum_logprob"].cpu().numpy().astype(np.float64) - want["sum_logprob"])
    assert np.all(err <= 1e-5 * (want["len"] + np.abs(want["sum_logprob"])) + 1e-12)


@pytest.mark.parametrize("by_slot", [False, True])
@pytest.mark.parametrize("gmax", [0, 2**30])
def test_hidden_callback_loop(cd, oracle, by_slot, gmax):
    V, H, B, steps = 3000, 128, 300, 8
    aut = wl.make_random_dfa(63, V, 20, 0.1, 0.15)
    dfa = cd.compile_dfa(aut.V, aut.S, aut.start, aut.row_ptr, aut.tok, aut.next, aut.accepting, device="cuda:0")
    dfa.set_head_gather_max(gmax)
    W = wl.make_head(63, V, H, 2.0, exact=True)
    hs = [wl.make_hidden(63, k, B, H, exact=True) for k in range(steps)]
    dev = [h.to("cuda:0") for h in hs]

    def next_hidden(step, row_ids, n_active):
        if not by_slot:
            return dev[step], False
        return dev[step].index_select(0, row_ids.long().clamp_(0, B - 1)), True

    got = cd.head_decode_loop_cb(dfa, next_hidden, W.to("cuda:0"), H, B, steps)
    torch.cuda.synchronize()
    want = oracle.head_decode_loop(aut, hs, W, H)
    for k in ("tokens", "len", "final_state", "done"):
        assert np.array_equal(got[k].cpu().numpy(), want[k]), k


def test_callback_failure_is_reported(cd):
    aut = wl.make_random_dfa(65, 512, 6, 0.2, 0.2)
    dfa = cd.compile_dfa(aut.V, aut.S, aut.start, aut.row_ptr, aut.tok, aut.next, aut.accepting, device="cuda:0")

    def bad(step, row_ids, n_active):
        raise RuntimeError("model forward failed")

    with pytest.raises(cd.CdError):
        cd.decode_loop_cb(dfa, bad, torch.float32, 8, 3)


def test_handle_level_limit_applies_to_every_loop(cd, oracle):
    """cd_set_limit (LIMIT early exit) on the device loop, the host-buffer loop, the
    callback loop and the LM-head loops, against the oracle's limited loop (O5).  Exact-arithmetic head
    inputs make the fp32 logits of a library matmul equal to the head's dot products."""
    V, H, B, steps = 2048, 128, 240, 8
    aut = wl.make_random_dfa(67, V, 16, 0.1, 0.3)
    acc = np.asarray(aut.accepting)
    sat = ((np.arange(aut.S) % 2 == 0) & (acc != 0)).astype(np.uint8)
    if sat.sum() == 0:
        sat = acc.astype(np.uint8)
    W = wl.make_head(67, V, H, 2.0, exact=True)
    hs = [wl.make_hidden(67, k, B, H, exact=True) for k in range(steps)]
    logits = [(h.double() @ W.double().t()).float().contiguous() for h in hs]  # exact in fp32
    full = oracle.decode_loop(aut, logits)
    n_sat = int(sum(1 for r in range(B) if full["done"][r] and sat[full["final_state"][r]]))
    assert n_sat >= 4
    limit = max(2, n_sat // 3)
    want = oracle.decode_loop(aut, logits, satisfying=sat, limit=limit, satisfied=0)
    assert (want["len"] < full["len"]).any()  # the limit really cancels rows

    dfa = cd.compile_dfa(aut.V, aut.S, aut.start, aut.row_ptr, aut.tok, aut.next, aut.accepting, device="cuda:0")
    dfa.set_satisfying(sat)
    ctr = torch.zeros(1, dtype=torch.int32, device="cuda:0")
    dfa.set_limit(limit, ctr)
    ldev = [x.to("cuda:0") for x in logits]
    hdev = [h.to("cuda:0") for h in hs]
    Wd = W.to("cuda:0")

    def check(got, name):
        torch.cuda.synchronize()
        for k in ("tokens", "len", "final_state", "done"):
            assert np.array_equal(got[k].cpu().numpy(), want[k]), (name, k)
        assert int(ctr) == want["satisfied"], name
        ctr.zero_()

    check(cd.decode_loop(dfa, ldev), "device loop")
    check(cd.decode_loop_host(dfa, [x.pin_memory() for x in logits]), "host loop")
    check(cd.decode_loop_cb(dfa, lambda k, ids, n: (ldev[k], False), torch.float32, B, steps), "callback loop")
    for gmax in (0, 2**30):
        dfa.set_head_gather_max(gmax)
        check(cd.head_decode_loop(dfa, hdev, Wd, H=H), f"head loop gmax={gmax}")
    check(cd.head_decode_loop_host(dfa, [h.pin_memory() for h in hs], Wd, H=H), "head host loop")
    check(cd.head_decode_loop_cb(dfa, lambda k, ids, n: (hdev[k], False), Wd, H, B, steps), "head callback loop")
    # a second batch of the same query starts with the counter already at the limit: nothing runs
    ctr.fill_(limit)
    got = cd.head_decode_loop(dfa, hdev, Wd, H=H)
    torch.cuda.synchronize()
    assert int(got["len"].max()) == 0 and int(got["done"].max()) == 0
    # cleared: the unlimited result again
    dfa.set_limit(0, None)
    got = cd.decode_loop(dfa, ldev)
    torch.cuda.synchronize()
    assert np.array_equal(got["tokens"].cpu().numpy(), full["tokens"])
