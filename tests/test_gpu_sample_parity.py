"""Parity of the sampled step (cd_set_sampling, through the C ABI) with the
oracle's O10.  The Gumbel-max decision is taken in fp32 on identical bits on both sides
(counter-based generator and fp32 operation sequence are part of the definition), so token,
state, done and histories are compared bit-exactly; logprob / lse within 1e-5*max(1,|ref|)."""
import numpy as np
import pytest
import torch

import workloads as wl

pytestmark = pytest.mark.gpu
TOL = 1e-5


@pytest.fixture(scope="module")
def cd():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    import paper_2606_31808_b200 as m

    m.lib()
    return m


@pytest.fixture(params=["dense", "gather_all", "gather_mixed"])
def mode(request):
    return request.param


def dev_dfa(cd, aut, mode):
    dfa = cd.compile_dfa(aut.V, aut.S, aut.start, aut.row_ptr, aut.tok, aut.next, aut.accepting, device="cuda:0")
    if mode == "gather_all":
        dfa.set_gather_max(2**30)
    elif mode == "gather_mixed":
        deg = torch.diff(torch.as_tensor(aut.row_ptr).cpu())
        deg = deg[deg > 0]
        dfa.set_gather_max(max(1, int(deg.median())))
    return dfa


def close(gpu, ref):
    gpu = np.asarray(gpu, np.float64)
    both_inf = np.isneginf(gpu) & np.isneginf(ref)
    err = np.abs(np.where(both_inf, 0.0, gpu - ref))
    return bool(np.all(err <= TOL * np.maximum(1.0, np.abs(np.where(both_inf, 0.0, ref)))))


def live_states(aut, n, mult=3):
    acc = np.asarray(aut.accepting)
    live = [s for s in range(aut.S) if not acc[s]]
    return [live[(i * mult) % len(live)] for i in range(n)]


@pytest.mark.parametrize("V,S,n,density,dtype,T", [
    (1000, 7, 37, 0.3, torch.float32, 1.0),
    (40000, 12, 70, 0.05, torch.bfloat16, 0.7),    # several tiles and units per row
    (262144, 16, 9, 0.02, torch.bfloat16, 1.3),    # full vocabulary, few rows: many units per row (merge path)
    (5000, 5, 300, 1.0, torch.bfloat16, 2.0),      # everything allowed: ties in y, noise decides
    (776, 4, 5, 0.5, torch.float32, 0.25),
])
def test_sampled_step_matches_oracle(cd, oracle, mode, V, S, n, density, dtype, T):
    aut = wl.make_random_dfa(51, V, S, density, 0.2)
    dfa = dev_dfa(cd, aut, mode)
    dfa.set_sampling(T, seed=0x1234567890ABCDEF, step_base=4)
    x = wl.make_logits(51, 0, n + 10, V, 2.0, dtype)
    states = live_states(aut, n)
    row_map = [(i * 7 + 3) % (n + 10) for i in range(n)]
    st_d = torch.tensor(states, dtype=torch.int32, device="cuda:0")
    rm_d = torch.tensor(row_map, dtype=torch.int32, device="cuda:0")
    tok, lp, lse, done = cd.step(dfa, x.to("cuda:0"), st_d, row_map=rm_d)
    torch.cuda.synchronize()
    o_tok, o_lp, o_lse, o_done, o_st = oracle.sample_step(aut, x, states, T, seed=0x1234567890ABCDEF, step=4,
                                                          row_map=row_map)
    assert tok.cpu().numpy().tolist() == o_tok.tolist()
    assert st_d.cpu().numpy().tolist() == o_st.tolist()
    assert done.cpu().numpy().tolist() == o_done.tolist()
    assert close(lp.cpu().numpy(), o_lp) and close(lse.cpu().numpy(), o_lse)
    # greedy is restored by temperature 0
    dfa.set_sampling(0.0)
    st_d = torch.tensor(states, dtype=torch.int32, device="cuda:0")
    tok, _, _, _ = cd.step(dfa, x.to("cuda:0"), st_d, row_map=rm_d)
    g_tok = oracle.step(aut, x, states, row_map=row_map)[0]
    assert tok.cpu().numpy().tolist() == g_tok.tolist()


def test_sampled_step_special_values(cd, oracle, mode):
    V, S, n = 600, 4, 20
    aut = wl.make_random_dfa(53, V, S, 0.3, 0.25)
    dfa = dev_dfa(cd, aut, mode)
    dfa.set_sampling(1.0, seed=7)
    x = wl.make_logits(53, 0, n, V, 2.0, torch.float32)
    lo, hi = int(aut.row_ptr[0]), int(aut.row_ptr[1])
    allowed0 = [int(t) for t in aut.tok[lo:hi]]
    x[0, allowed0] = float("-inf")      # every allowed logit -inf: lowest allowed id, logprob -inf
    x[1, allowed0[:3]] = float("nan")   # NaN read as -inf
    x[2, :] = 1e30                      # huge everywhere
    x[3, [t for t in range(V) if t not in set(allowed0)]] = float("nan")  # poisoned complement
    states = [0] * n
    st_d = torch.tensor(states, dtype=torch.int32, device="cuda:0")
    tok, lp, lse, done = cd.step(dfa, x.to("cuda:0"), st_d)
    torch.cuda.synchronize()
    o_tok, o_lp, o_lse, o_done, o_st = oracle.sample_step(aut, x, states, 1.0, seed=7)
    assert tok.cpu().numpy().tolist() == o_tok.tolist() and st_d.cpu().numpy().tolist() == o_st.tolist()
    assert close(lp.cpu().numpy(), o_lp) and close(lse.cpu().numpy(), o_lse)
    assert tok[0] == allowed0[0] and np.isneginf(float(lp[0]))


@pytest.mark.parametrize("kind,V,B,steps,dtype", [("dfa", 3000, 300, 8, torch.bfloat16), ("trie", 2000, 150, 5, torch.float32)])
def test_sampled_decode_loop_matches_oracle(cd, oracle, mode, kind, V, B, steps, dtype):
    if kind == "dfa":
        aut = wl.make_random_dfa(57, V, 20, 0.1, 0.15)
    else:
        aut = wl.make_trie(V, wl.draw_labels(57, V, 25, 1, 5))
    dfa = dev_dfa(cd, aut, mode)
    dfa.set_sampling(0.9, seed=99, step_base=2)
    logits = [wl.make_logits(57, k, B, V, 2.0, dtype) for k in range(steps)]
    got = cd.decode_loop(dfa, [x.to("cuda:0") for x in logits])
    torch.cuda.synchronize()
    want = oracle.sample_decode_loop(aut, logits, 0.9, seed=99, step_base=2)
    for k in ("tokens", "len", "final_state", "done"):
        assert np.array_equal(got[k].cpu().numpy(), want[k]), k
    slp = got["sum_logprob"].cpu().numpy().astype(np.float64)
    assert np.all(np.abs(slp - want["sum_logprob"]) <= TOL * (want["len"] + np.abs(want["sum_logprob"])) + 1e-12)
    # same seed reproduces bit for bit; another seed does not
    again = cd.decode_loop(dfa, [x.to("cuda:0") for x in logits])
    assert torch.equal(again["tokens"], got["tokens"]) and torch.equal(again["sum_logprob"], got["sum_logprob"])
    dfa.set_sampling(0.9, seed=100, step_base=2)
    other = cd.decode_loop(dfa, [x.to("cuda:0") for x in logits])
    assert not torch.equal(other["tokens"], got["tokens"])


def test_sampled_full_size_c4_batch(cd, oracle):
    """One c4 step at full size (n = 4096, V = 262144, the launch configuration bench.py times) with
    sampling on: EVERY row compared with the oracle, bit for bit (the oracle touches only the allowed
    logits of a row, so all 4096 rows cost about a second)."""
    cfg = wl.CONFIGS["c4"]
    aut = wl.build_automaton(cfg)
    dfa = cd.compile_dfa(aut.V, aut.S, aut.start, aut.row_ptr, aut.tok, aut.next, aut.accepting, device="cuda:0")
    dfa.set_sampling(1.0, seed=2026, step_base=0)
    x = wl.make_logits(cfg.seed, 0, cfg.B, cfg.V, cfg.std, cfg.dtype, device="cuda:0")
    states = live_states(aut, cfg.B, mult=7)
    st_d = torch.tensor(states, dtype=torch.int32, device="cuda:0")
    tok, lp, lse, done = cd.step(dfa, x, st_d)
    torch.cuda.synchronize()
    # the noise is keyed by the ORIGINAL row id = logits row, so the host copy keeps the row positions
    host = x.cpu()
    o_tok, o_lp, o_lse, o_done, o_st = oracle.sample_step(aut, host, states, 1.0, seed=2026, step=0)
    assert tok.cpu().numpy().tolist() == o_tok.tolist()
    assert st_d.cpu().numpy().tolist() == o_st.tolist()
    assert done.cpu().numpy().tolist() == o_done.tolist()
    assert close(lp.cpu().numpy(), o_lp) and close(lse.cpu().numpy(), o_lse)
    # and a whole sampled c4-shaped loop of 4 steps over all 4096 rows, both loop modes
    xs = [x, wl.make_logits(cfg.seed, 1, cfg.B, cfg.V, cfg.std, cfg.dtype, device="cuda:0")]
    steps = [xs[k & 1] for k in range(4)]
    hosts = [host, xs[1].cpu()]
    want = oracle.sample_decode_loop(aut, [hosts[k & 1] for k in range(4)], 1.0, seed=2026)
    for lm in (cd.LOOP_AUTO, cd.LOOP_BARRIER, cd.LOOP_PER_STEP):
        dfa.set_loop_mode(lm)
        got = cd.decode_loop(dfa, steps)
        for k in ("tokens", "len", "final_state", "done"):
            assert np.array_equal(got[k].cpu().numpy(), want[k]), (lm, k)
    dfa.close()


# ---------------------------------------------------------------- an independent check of the sampled token
# The oracle's O10 restates the generator and its fp32 logarithm operation by operation, so bit-exact parity with it
# does not by itself rule out a mistake both sides share.  Here the decision is recomputed a third way: the uniform
# u of (seed, row, step, token) from a numpy statement of the counter hash (held against murmur3's published
# finalizer vectors below), g = -log(-log u) with libm in float64, t* = argmax over the allowed set of y_t + g_t.
# Wherever the winner leads the runner-up by more than the fp32 error of the kernel's y + g (the logarithm's 3e-7
# relative error twice over, |g| <= 17, one rounding of the sum: < 1e-5) the GPU token must be that argmax.
def _np_fmix32(h):
    h = h.astype(np.uint64)
    h ^= h >> np.uint64(16)
    h = (h * np.uint64(0x85EBCA6B)) & np.uint64(0xFFFFFFFF)
    h ^= h >> np.uint64(13)
    h = (h * np.uint64(0xC2B2AE35)) & np.uint64(0xFFFFFFFF)
    h ^= h >> np.uint64(16)
    return h


def _np_uniform(seed, row, step, toks):
    M = np.uint64(0xFFFFFFFF)
    lo, hi = np.uint64(seed & 0xFFFFFFFF), np.uint64(seed >> 32)
    h = _np_fmix32(np.array([lo ^ ((np.uint64(row) * np.uint64(0x9E3779B1)) & M)]))
    rk = _np_fmix32(h ^ ((np.uint64(step) * np.uint64(0x85EBCA77)) & M) ^ hi)
    t = toks.astype(np.uint64)
    hh = _np_fmix32((_np_fmix32(rk ^ ((t * np.uint64(0xC2B2AE3D)) & M)) + np.uint64(0x27D4EB2F)) & M)
    return (2.0 * (hh >> np.uint64(9)).astype(np.float64) + 1.0) * 2.0**-24


def test_numpy_generator_is_the_published_finalizer_and_the_oracles_uniform(oracle):
    got = _np_fmix32(np.array([0, 1, 0xFFFFFFFF], dtype=np.uint64)).tolist()
    assert got == [0x00000000, 0x514E28B7, 0x81F16F39]  # murmur3_32 of the empty key, seeds 0, 1, 0xFFFFFFFF
    toks = np.arange(0, 3000, 7)
    u = _np_uniform(0x1234567890ABCDEF, 77, 5, toks)
    g = np.array([oracle.gumbel(0x1234567890ABCDEF, 77, 5, int(t)) for t in toks])
    assert np.all(np.abs(-np.log(-np.log(u)) - g) <= 1e-5)


@pytest.mark.parametrize("V,S,n,density,dtype,T", [
    (40000, 12, 70, 0.05, torch.bfloat16, 0.7),
    (262144, 16, 24, 0.02, torch.bfloat16, 1.3),
    (5000, 5, 300, 1.0, torch.float32, 2.0),
])
def test_sampled_token_is_the_float64_gumbel_argmax(cd, mode, V, S, n, density, dtype, T):
    seed, step = 0x0FEDCBA987654321, 9
    aut = wl.make_random_dfa(52, V, S, density, 0.2)
    dfa = dev_dfa(cd, aut, mode)
    dfa.set_sampling(T, seed=seed, step_base=step)
    x = wl.make_logits(52, 0, n + 10, V, 2.0, dtype)
    states = live_states(aut, n)
    row_map = [(i * 7 + 3) % (n + 10) for i in range(n)]
    st_d = torch.tensor(states, dtype=torch.int32, device="cuda:0")
    tok, _, _, _ = cd.step(dfa, x.to("cuda:0"), st_d, row_map=torch.tensor(row_map, dtype=torch.int32, device="cuda:0"))
    tok = tok.cpu().numpy()
    rp, tk = np.asarray(aut.row_ptr), np.asarray(aut.tok)
    inv_T = np.float32(1.0) / np.float32(T)
    decided = 0
    for i in range(n):
        A = tk[rp[states[i]]:rp[states[i] + 1]].astype(np.int64)
        y = (x[row_map[i]].float().numpy()[A] * inv_T).astype(np.float64)  # y_t = fl32(x_t * fl32(1 / T))
        score = y - np.log(-np.log(_np_uniform(seed, row_map[i], step, A)))
        order = np.argsort(-score, kind="stable")
        lead = score[order[0]] - score[order[1]] if A.size > 1 else np.inf
        assert int(tok[i]) in set(A.tolist())
        if lead > 1e-5 * max(1.0, abs(score[order[0]])):
            decided += 1
            assert int(tok[i]) == int(A[order[0]]), (i, int(tok[i]), int(A[order[0]]), lead)
        else:  # a near tie: either of the two leaders
            assert int(tok[i]) in (int(A[order[0]]), int(A[order[1]]))
    assert decided >= 0.95 * n  # the check is not vacuous
    dfa.close()
