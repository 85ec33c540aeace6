"""What a handle's scratch memory carries from one loop to the next (round-2 review findings).

- The batch grows on one handle and stream: the step buffers are replaced and their launch generation
  restarts, while the queue ring of the whole-loop kernel is tagged with generations.  A ring that survived
  the regrowth would hand the next loop stale entries as if they were published.
- Two whole-loop launches on two streams at once: each needs every one of its thread blocks to run, so they
  must be ordered, not interleaved, or they starve each other until the idle timeout.
Both against the oracle, bit for bit in tokens / lengths / states / done flags.
"""
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


def _same(out, want, tag):
    for k in ("tokens", "len", "final_state", "done"):
        assert np.array_equal(out[k].cpu().numpy(), want[k]), (tag, k)
    g, r = out["sum_logprob"].cpu().numpy().astype(np.float64), want["sum_logprob"]
    fin = np.isfinite(r)
    assert np.array_equal(np.isfinite(g), fin), tag
    assert np.all(np.abs(g[fin] - r[fin]) <= 1e-5 * np.maximum(1.0, want["len"][fin] + np.abs(r[fin]))), tag


@pytest.mark.parametrize("sizes", [(10, 20), (3000, 4000), (1, 2, 3, 70, 700)])
@pytest.mark.parametrize("mode", ["dense", "gather_all"])
def test_batch_grows_on_one_handle_and_stream(cd, oracle, sizes, mode):
    base = wl.scaled(wl.CONFIGS["c3"], V=20000, B=sizes[0], S=40, max_steps=6)
    aut = wl.build_automaton(base)
    dfa = cd.compile_dfa(aut.V, aut.S, aut.start, aut.row_ptr, aut.tok, aut.next, aut.accepting, device="cuda:0")
    if mode == "gather_all":
        dfa.set_gather_max(2**30)
    for B in sizes:
        cfg = wl.scaled(wl.CONFIGS["c3"], V=20000, B=B, S=40, max_steps=6)
        xs = wl.build_step_logits(cfg, aut, device="cuda:0", batch=B)
        want = oracle.decode_loop(aut, [x.cpu() for x in xs])
        for rep in range(3):  # several launches per size: the ring holds entries of generations 1, 2, 3 when B grows
            _same(cd.decode_loop(dfa, xs), want, (B, rep))
    dfa.close()


def test_two_loops_in_flight_on_two_streams(cd, oracle):
    cfg = wl.scaled(wl.CONFIGS["c3"], V=65536, B=256, S=64, max_steps=8)
    aut = wl.build_automaton(cfg)
    dfa = cd.compile_dfa(aut.V, aut.S, aut.start, aut.row_ptr, aut.tok, aut.next, aut.accepting, device="cuda:0")
    la = wl.build_step_logits(cfg, aut, device="cuda:0", batch=0)
    lb = wl.build_step_logits(cfg, aut, device="cuda:0", batch=1)
    want = {"a": oracle.decode_loop(aut, [x.cpu() for x in la]), "b": oracle.decode_loop(aut, [x.cpu() for x in lb])}
    torch.cuda.synchronize()
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    for rep in range(20):
        # both enqueued before either is waited for: without ordering the second launch starts while the first runs
        with torch.cuda.stream(s1):
            oa = cd.decode_loop_async(dfa, la)
        with torch.cuda.stream(s2):
            ob = cd.decode_loop_async(dfa, lb)
        with torch.cuda.stream(s2):
            cd.loop_sync(dfa)
        with torch.cuda.stream(s1):
            cd.loop_sync(dfa)
        _same(oa, want["a"], ("a", rep))
        _same(ob, want["b"], ("b", rep))
    dfa.close()
