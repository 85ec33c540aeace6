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
