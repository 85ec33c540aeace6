"""Seeded fuzz of the CUDA path against the oracle: random shapes (vocabulary sizes off every tile /
word boundary, strides with padding, row_map with repeats, dense and sparse automata, tries), random
modes (dense / gathered / mixed, greedy / sampled, logits / LM head), one step and whole loops.
Same bars as everywhere: bit-exact integers, 1e-5*max(1,|ref|) for log-probs (head path on
exact-arithmetic inputs)."""
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


def close(gpu, ref, tol=TOL):
    gpu = np.asarray(gpu, np.float64)
    ref = np.asarray(ref, np.float64)
    both_inf = np.isneginf(gpu) & np.isneginf(ref)
    with np.errstate(invalid="ignore"):
        err = np.abs(np.where(both_inf, 0.0, gpu - ref))
    return bool(np.all(err <= tol * np.maximum(1.0, np.abs(np.where(both_inf, 0.0, ref)))))


def random_case(rng, max_V=70000):
    kind = rng.choice(["dfa", "dfa", "trie"])
    V = int(rng.choice([rng.integers(40, 3000), rng.integers(3000, max_V)]))
    if kind == "dfa":
        S = int(rng.integers(2, 40))
        density = float(rng.choice([0.002, 0.02, 0.2, 0.7, 1.0]))
        aut = wl.make_random_dfa(int(rng.integers(1 << 30)), V, S, density, float(rng.choice([0.0, 0.1, 0.4])))
    else:
        K = int(rng.integers(1, 30))
        aut = wl.make_trie(V, wl.draw_labels(int(rng.integers(1 << 30)), V, K, 1, int(rng.integers(1, 5))))
    return aut, V


def set_mode(dfa, aut, rng):
    mode = rng.choice(["dense", "gather_all", "mixed", "auto"])
    if mode == "gather_all":
        dfa.set_gather_max(2**30)
    elif mode == "mixed":
        deg = torch.diff(torch.as_tensor(aut.row_ptr))
        deg = deg[deg > 0]
        dfa.set_gather_max(max(1, int(deg.median())))
    elif mode == "auto":
        dfa.set_gather_max(-1)
    return mode


@pytest.mark.parametrize("seed", range(24))
def test_fuzz_step(cd, oracle, seed):
    rng = np.random.default_rng(1000 + seed)
    aut, V = random_case(rng)
    dtype = [torch.float32, torch.bfloat16][int(rng.integers(2))]
    align = 4 if dtype == torch.float32 else 8
    ld = (V + align - 1) // align * align + align * int(rng.integers(0, 3))
    rows = int(rng.integers(1, 200))
    n = int(rng.integers(1, 260))
    dfa = cd.compile_dfa(aut.V, aut.S, aut.start, aut.row_ptr, aut.tok, aut.next, aut.accepting, device="cuda:0")
    mode = set_mode(dfa, aut, rng)
    sample = bool(rng.integers(2))
    T, rseed, sb = float(rng.choice([0.5, 1.0, 3.0])), int(rng.integers(1 << 62)), int(rng.integers(0, 50))
    if sample:
        dfa.set_sampling(T, seed=rseed, step_base=sb)
    x = wl.make_logits(seed, 0, rows, V, float(rng.choice([0.5, 2.0, 6.0])), dtype, ld=ld)
    states = [int(s) for s in rng.integers(0, aut.S, n)]       # includes accepting states
    row_map = [int(r) for r in rng.integers(0, rows, n)]       # with repeats
    st_d = torch.tensor(states, dtype=torch.int32, device="cuda:0")
    rm_d = torch.tensor(row_map, dtype=torch.int32, device="cuda:0")
    tok, lp, lse, done = cd.step(dfa, x.to("cuda:0"), st_d, row_map=rm_d)
    torch.cuda.synchronize()
    if sample:
        o_tok, o_lp, o_lse, o_done, o_st = oracle.sample_step(aut, x, states, T, seed=rseed, step=sb, row_map=row_map)
    else:
        o_tok, o_lp, o_lse, o_done, o_st = oracle.step(aut, x, states, row_map=row_map)
    ctx = (seed, mode, sample, V, aut.S, n, str(dtype))
    assert tok.cpu().numpy().tolist() == o_tok.tolist(), ctx
    assert st_d.cpu().numpy().tolist() == o_st.tolist(), ctx
    assert done.cpu().numpy().tolist() == o_done.tolist(), ctx
    assert close(lp.cpu().numpy(), o_lp) and close(lse.cpu().numpy(), o_lse), ctx


@pytest.mark.parametrize("seed", range(12))
def test_fuzz_loop(cd, oracle, seed):
    rng = np.random.default_rng(2000 + seed)
    aut, V = random_case(rng, max_V=20000)
    dtype = [torch.float32, torch.bfloat16][int(rng.integers(2))]
    B, steps = int(rng.integers(1, 400)), int(rng.integers(1, 9))
    dfa = cd.compile_dfa(aut.V, aut.S, aut.start, aut.row_ptr, aut.tok, aut.next, aut.accepting, device="cuda:0")
    mode = set_mode(dfa, aut, rng)
    sample = bool(rng.integers(2))
    if sample:
        dfa.set_sampling(0.9, seed=seed, step_base=1)
    align = 4 if dtype == torch.float32 else 8
    ld = (V + align - 1) // align * align
    logits = [wl.make_logits(seed, k, B, V, 2.0, dtype, ld=ld) for k in range(steps)]
    got = cd.decode_loop(dfa, [x.to("cuda:0") for x in logits])
    torch.cuda.synchronize()
    want = oracle.sample_decode_loop(aut, logits, 0.9, seed=seed, step_base=1) if sample else oracle.decode_loop(aut, logits)
    for k in ("tokens", "len", "final_state", "done"):
        assert np.array_equal(got[k].cpu().numpy(), want[k]), (k, seed, mode, sample)
    slp = got["sum_logprob"].cpu().numpy().astype(np.float64)
    fin = np.isfinite(want["sum_logprob"])
    assert np.all(np.abs(slp[fin] - want["sum_logprob"][fin]) <= TOL * (want["len"][fin] + np.abs(want["sum_logprob"][fin])) + 1e-12)


@pytest.mark.parametrize("seed", range(12))
def test_fuzz_head_step(cd, oracle, seed):
    rng = np.random.default_rng(3000 + seed)
    aut, V = random_case(rng, max_V=6000)
    H = 8 * int(rng.integers(1, 40))
    rows, n = int(rng.integers(1, 300)), int(rng.integers(1, 300))
    dfa = cd.compile_dfa(aut.V, aut.S, aut.start, aut.row_ptr, aut.tok, aut.next, aut.accepting, device="cuda:0")
    gm = int(rng.choice([0, 2**30, -1, 5]))
    dfa.set_head_gather_max(gm)
    sample = bool(rng.integers(2))
    if sample:
        dfa.set_sampling(1.2, seed=seed + 5, step_base=2)
    hid = wl.make_hidden(seed, 0, rows, H, exact=True, ld=H + 8 * int(rng.integers(0, 3)))
    W = wl.make_head(seed, V, H, 2.0, exact=True, ld=H + 8 * int(rng.integers(0, 3)))
    states = [int(s) for s in rng.integers(0, aut.S, n)]
    row_map = [int(r) for r in rng.integers(0, rows, n)]
    st_d = torch.tensor(states, dtype=torch.int32, device="cuda:0")
    rm_d = torch.tensor(row_map, dtype=torch.int32, device="cuda:0")
    tok, lp, lse, done = cd.head_step(dfa, hid.to("cuda:0"), W.to("cuda:0"), st_d, row_map=rm_d, H=H)
    torch.cuda.synchronize()
    if sample:
        x32 = (hid[:, :H].double() @ W[:, :H].double().t()).float().contiguous()  # exact in fp32
        o_tok, o_lp, o_lse, o_done, o_st = oracle.sample_step(aut, x32, states, 1.2, seed=seed + 5, step=2, row_map=row_map)
    else:
        o_tok, o_lp, o_lse, o_done, o_st, _ = oracle.head_step(aut, hid, W, H, states, row_map=row_map)
    ctx = (seed, gm, sample, V, H, aut.S, n)
    assert tok.cpu().numpy().tolist() == o_tok.tolist(), ctx
    assert st_d.cpu().numpy().tolist() == o_st.tolist() and done.cpu().numpy().tolist() == o_done.tolist(), ctx
    assert close(lp.cpu().numpy(), o_lp) and close(lse.cpu().numpy(), o_lse), ctx
