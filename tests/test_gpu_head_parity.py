"""Parity of cd_head_step (through the C ABI) with the oracle's O6.

Two kinds of inputs:
  * exact-arithmetic inputs (workloads.make_hidden / make_head with exact=True: multiples
    of 1/8): every partial sum of every dot product is exactly representable in fp32, so
    the logits do not depend on the accumulation order of the tensor cores and the bar is
    the same as for cd_step -- bit-exact token / state / done (ties included: logits are
    multiples of 1/64, so equal maxima are frequent), logprob / lse within 1e-5;
  * gaussian inputs: the kernel's fp32 accumulation differs from the oracle's double by at
    most EPS_X per logit ((H/16 + 40) additions of relative error
    2^-23 on partial sums bounded by sum_h |a_h||w_h|).  Where the oracle's best allowed
    logit leads the runner-up by more than 2*EPS_X the token must match; otherwise the GPU
    token must be an allowed token whose oracle logit is within 2*EPS_X of the best, and
    state / done must follow from that token.  logprob / lse: 1e-5*max(1,|ref|) + 2*EPS_X.

Each test runs with every state gathered, every state dense (tcgen05 contraction) and the
automatic mix.
"""
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


@pytest.fixture(params=["gather", "dense", "mixed"])
def mode(request):
    return request.param


def dev_dfa(cd, aut, mode):
    dfa = cd.compile_dfa(aut.V, aut.S, aut.start, aut.row_ptr, aut.tok, aut.next, aut.accepting, device="cuda:0")
    if mode == "gather":
        dfa.set_head_gather_max(2**30)
    elif mode == "dense":
        dfa.set_head_gather_max(0)
    else:
        deg = torch.diff(torch.as_tensor(aut.row_ptr).cpu())
        deg = deg[deg > 0]
        dfa.set_head_gather_max(max(1, int(deg.median())) if deg.numel() else 1)
    return dfa


def eps_x(hid, W, H):
    """Bound of |fp32-accumulated logit - exact logit| for these operands."""
    a = hid[:, :H].abs().to(torch.float64).max(dim=0).values  # per-h max over rows
    A = 0.0  # >= sum_h |a_h||w_h| for every (row, token)
    for t0 in range(0, W.shape[0], 16384):
        A = max(A, float((W[t0:t0 + 16384, :H].abs().to(torch.float64) @ a).max()))
    return (H / 16 + 40) * 2.0**-23 * A


def transitions(aut):
    rp, tk, nx = (np.asarray(x) for x in (aut.row_ptr, aut.tok, aut.next))
    d = {}
    for s in range(aut.S):
        for j in range(int(rp[s]), int(rp[s + 1])):
            d[(s, int(tk[j]))] = int(nx[j])
    return d


def run_case(cd, oracle, aut, dfa, hid, W, H, states, row_map=None, exact=True, check=None, W_dev=None):
    """GPU on every slot; the oracle on the slots listed in `check` (default: all)."""
    dev = "cuda:0"
    hid_d, W_d = hid.to(dev), (W.to(dev) if W_dev is None else W_dev)
    st_d = torch.tensor(states, dtype=torch.int32, device=dev)
    rm_d = None if row_map is None else torch.tensor(row_map, dtype=torch.int32, device=dev)
    tok, lp, lse, done = cd.head_step(dfa, hid_d, W_d, st_d, row_map=rm_d, H=H)
    torch.cuda.synchronize()
    tok, lp, lse, done, st_new = (t.cpu().numpy() for t in (tok, lp, lse, done, st_d))
    if check is not None:
        check = list(check)
        tok, lp, lse, done, st_new = (x[check] for x in (tok, lp, lse, done, st_new))
        row_map = [(i if row_map is None else row_map[i]) for i in check]
        states = [states[i] for i in check]
    o_tok, o_lp, o_lse, o_done, o_st, gap = oracle.head_step(aut, hid, W, H, states, row_map=row_map)
    n = len(states)
    if exact:
        assert tok.tolist() == o_tok.tolist()
        assert st_new.tolist() == o_st.tolist()
        assert done.tolist() == o_done.tolist()
        ex = 0.0
    else:
        ex = 2.0 * eps_x(hid, W, H)
        delta = transitions(aut)
        acc = np.asarray(aut.accepting)
        n_flip = 0
        for i in range(n):
            if tok[i] == o_tok[i]:
                assert st_new[i] == o_st[i] and done[i] == o_done[i]
                continue
            n_flip += 1
            assert gap[i] <= ex, (i, gap[i], ex)
            r = i if row_map is None else row_map[i]
            key = (states[i], int(tok[i]))
            assert key in delta  # an allowed token
            best = oracle.head_logit(hid, W, H, r, int(o_tok[i]))
            mine = oracle.head_logit(hid, W, H, r, int(tok[i]))
            assert best - mine <= ex
            assert st_new[i] == delta[key] and done[i] == acc[delta[key]]
        assert n_flip <= max(2, n // 10)
    for g, r in ((lp, o_lp), (lse, o_lse)):
        g = g.astype(np.float64)
        both_inf = np.isneginf(g) & np.isneginf(r)
        err = np.abs(np.where(both_inf, 0.0, g - r))
        bound = TOL * np.maximum(1.0, np.abs(np.where(both_inf, 0.0, r))) + ex
        assert np.all(err <= bound), (float(err.max()), float(bound.min()))
    if not exact:  # empirical sanity: the typical error is far below the worst-case bound
        e = np.abs(lse.astype(np.float64) - o_lse)
        e = e[np.isfinite(e)]
        assert e.size == 0 or float(np.sqrt(np.mean(e**2))) <= 2e-5 * max(1.0, float(np.abs(o_lse[np.isfinite(o_lse)]).max()))
    return tok, st_new


def live_states(aut, n, mult=3):
    acc = np.asarray(aut.accepting)
    live = [s for s in range(aut.S) if not acc[s]]
    return [live[(i * mult) % len(live)] for i in range(n)]


@pytest.mark.parametrize("V,H,S,n,density", [
    (1000, 64, 7, 37, 0.3),      # one row tile, V tail inside the 4th vocabulary tile
    (1000, 200, 7, 130, 0.3),    # K tail (200 = 3*64 + 8), two row tiles with a ragged second
    (5000, 256, 40, 300, 0.05),  # 20 vocabulary tiles, 3 row tiles
    (4096, 128, 16, 128, 1.0),   # everything allowed
    (777, 72, 5, 5, 0.5),
])
def test_exact_inputs_bit_exact(cd, oracle, mode, V, H, S, n, density):
    aut = wl.make_random_dfa(11, V, S, density, 0.2)
    dfa = dev_dfa(cd, aut, mode)
    hid = wl.make_hidden(11, 0, n, H, exact=True, ld=H + 8)
    W = wl.make_head(11, V, H, 2.0, exact=True, ld=H + 16)
    run_case(cd, oracle, aut, dfa, hid, W, H, live_states(aut, n))


def test_ties_across_tile_boundaries(cd, oracle, mode):
    V, H, S, n = 2048, 64, 3, 140
    aut = wl.make_random_dfa(5, V, S, 1.0, 0.3)
    dfa = dev_dfa(cd, aut, mode)
    hid = wl.make_hidden(5, 0, n, H, exact=True)
    W = wl.make_head(5, V, H, 2.0, exact=True)
    # identical rows with the largest possible dot product sit on both sides of 32-column,
    # tile (256) and range boundaries: the lowest id must win
    big = torch.sign(hid[0, :H].float()).to(torch.bfloat16)  # maximises <hid[0], w>
    for t in (1791, 1792, 1023, 1024, 511, 512, 287, 288):
        W[t, :H] = big
    tok, _ = run_case(cd, oracle, aut, dfa, hid, W, H, live_states(aut, n))
    assert tok[0] == 287


def test_row_map_and_accepting_slots(cd, oracle, mode):
    V, H, S, n = 1500, 128, 9, 70
    aut = wl.make_random_dfa(13, V, S, 0.2, 0.3)
    dfa = dev_dfa(cd, aut, mode)
    hid = wl.make_hidden(13, 0, 200, H, exact=True)
    W = wl.make_head(13, V, H, 2.0, exact=True)
    states = [(i * 5) % S for i in range(n)]  # includes accepting states: those slots never advance
    row_map = [(i * 37 + 11) % 200 for i in range(n)]
    run_case(cd, oracle, aut, dfa, hid, W, H, states, row_map=row_map)


def test_trie_states(cd, oracle, mode):
    V, H, n = 3000, 192, 90
    labels = wl.draw_labels(2, V, 20, 1, 4)
    aut = wl.make_trie(V, labels)
    dfa = dev_dfa(cd, aut, mode)
    hid = wl.make_hidden(2, 1, n, H, exact=True)
    W = wl.make_head(2, V, H, 2.0, exact=True)
    run_case(cd, oracle, aut, dfa, hid, W, H, live_states(aut, n, mult=1))


@pytest.mark.parametrize("V,H,S,n,density", [(3000, 256, 12, 150, 0.1), (1024, 2560, 4, 40, 0.5)])
def test_gaussian_inputs_within_accumulation_error(cd, oracle, mode, V, H, S, n, density):
    aut = wl.make_random_dfa(17, V, S, density, 0.2)
    dfa = dev_dfa(cd, aut, mode)
    hid = wl.make_hidden(17, 0, n, H)
    W = wl.make_head(17, V, H, 2.0)
    run_case(cd, oracle, aut, dfa, hid, W, H, live_states(aut, n), exact=False)


def test_nan_and_inf_embeddings(cd, oracle, mode):
    V, H, S, n = 600, 64, 4, 33
    aut = wl.make_random_dfa(19, V, S, 0.3, 0.25)
    dfa = dev_dfa(cd, aut, mode)
    hid = wl.make_hidden(19, 0, n, H, exact=True)
    W = wl.make_head(19, V, H, 2.0, exact=True)
    lo, hi = int(aut.row_ptr[0]), int(aut.row_ptr[1])
    allowed0 = [int(t) for t in aut.tok[lo:hi]]
    W[allowed0[0], 3] = float("nan")      # an allowed NaN logit is read as -inf (G6)
    for t in range(V):                     # poisoned complement of state 0
        if t not in set(allowed0) and t % 7 == 0:
            W[t, 5] = float("nan")
    states = [0] * n
    run_case(cd, oracle, aut, dfa, hid, W, H, states)


def test_arguments(cd):
    aut = wl.make_random_dfa(1, 256, 3, 0.5, 0.3)
    dfa = cd.compile_dfa(aut.V, aut.S, aut.start, aut.row_ptr, aut.tok, aut.next, aut.accepting, device="cuda:0")
    hid = torch.zeros((4, 60), dtype=torch.bfloat16, device="cuda:0")
    W = torch.zeros((256, 60), dtype=torch.bfloat16, device="cuda:0")
    st = torch.zeros(4, dtype=torch.int32, device="cuda:0")
    with pytest.raises(cd.CdError):
        cd.head_step(dfa, hid, W, st, H=60)  # H not a multiple of 8
    hid = torch.zeros((4, 64), dtype=torch.bfloat16, device="cuda:0")
    W = torch.zeros((256, 64), dtype=torch.bfloat16, device="cuda:0")
    tok, lp, lse, done = cd.head_step(dfa, hid, W, st, n=0)  # n == 0 launches nothing
    # all-zero logits: lowest allowed id, logprob = -log(deg)
    tok, lp, lse, done = cd.head_step(dfa, hid, W, st)
    torch.cuda.synchronize()
    deg = int(aut.row_ptr[1] - aut.row_ptr[0])
    assert tok.cpu().tolist() == [int(aut.tok[0])] * 4
    assert abs(float(lp[0]) + np.log(deg)) < 1e-5


# ---------------------------------------------------------------- full size (V = 262144, H = 2560)
@pytest.fixture(scope="module")
def full_head():
    """Output embedding of the bench configuration, exact and gaussian, on both sides."""
    V, H = 262144, 2560
    out = {}
    for kind, exact in (("exact", True), ("gauss", False)):
        Wd = wl.make_head(7, V, H, 2.0, device="cuda:0", exact=exact)
        out[kind] = (Wd, Wd.cpu())
    return V, H, out


@pytest.mark.parametrize("kind", ["exact", "gauss"])
@pytest.mark.parametrize("name,n_check", [("c2", 1024), ("c3", 512), ("c4", 1024)])
def test_full_size_configs(cd, oracle, full_head, kind, name, n_check):
    """BASELINE.json configs c2-c4 at full size in the launch configuration bench.py times
    (automatic gather threshold): every row on the GPU; the oracle (double-precision dot products,
    ~3-13 ms per row) on EVERY row of c2 and c3 and on 1024 evenly spaced rows of c4 (rows are
    independent)."""
    V, H, Ws = full_head
    W_dev, W_cpu = Ws[kind]
    cfg = wl.CONFIGS[name]
    aut = wl.build_automaton(cfg)
    dfa = cd.compile_dfa(aut.V, aut.S, aut.start, aut.row_ptr, aut.tok, aut.next, aut.accepting, device="cuda:0")
    n = cfg.B
    hid = wl.make_hidden(cfg.seed, 0, n, H, exact=(kind == "exact"))
    if cfg.kind == "dfa":
        states = live_states(aut, n, mult=7)
    else:
        states = live_states(aut, n, mult=1)  # every trie node, root included
    check = sorted(set(int(i) for i in np.linspace(0, n - 1, n_check).astype(int)))
    run_case(cd, oracle, aut, dfa, hid, W_cpu, H, states, exact=(kind == "exact"), check=check, W_dev=W_dev)


@pytest.mark.parametrize("kind", ["exact", "gauss"])
@pytest.mark.parametrize("n,gathered", [(14, True), (36, True), (64, False)])
def test_late_step_of_c3_few_rows_of_big_states(cd, oracle, full_head, kind, n, gathered):
    """A late step of an early-exit loop on c3 (V = 262144, states of ~5243 transitions): with the automatic
    policy a handful of rows is GATHERED -- every row cut into 41 pieces over as many CTAs, merged by
    head_gather_finish_kernel -- as long as the rows together touch fewer than 0.8 V rows of W; above, the dense
    contraction runs.  Every row against the oracle, and the automatic result against the forced dense and forced
    gather ones (tokens / states identical on exact inputs)."""
    V, H, Ws = full_head
    W_dev, W_cpu = Ws[kind]
    cfg = wl.CONFIGS["c3"]
    aut = wl.build_automaton(cfg)
    deg = np.diff(np.asarray(aut.row_ptr))
    states = live_states(aut, n, mult=7)
    assert (float(deg[states].sum()) < 0.8 * V) == gathered  # which side of the policy this case is on
    hid = wl.make_hidden(cfg.seed, 5, n, H, exact=(kind == "exact"))
    dfa = cd.compile_dfa(aut.V, aut.S, aut.start, aut.row_ptr, aut.tok, aut.next, aut.accepting, device="cuda:0")
    run_case(cd, oracle, aut, dfa, hid, W_cpu, H, states, exact=(kind == "exact"), W_dev=W_dev)
    if kind == "exact":
        res = []
        for g in (-1, 0, 2**30):
            dfa.set_head_gather_max(g)
            st = torch.tensor(states, dtype=torch.int32, device="cuda:0")
            tok, lp, lse, done = cd.head_step(dfa, hid.to("cuda:0"), W_dev, st, H=H)
            res.append((tok.cpu(), st.cpu(), done.cpu(), lse.cpu()))
        for r in res[1:]:
            assert torch.equal(res[0][0], r[0]) and torch.equal(res[0][1], r[1]) and torch.equal(res[0][2], r[2])
            assert torch.allclose(res[0][3], r[3], rtol=0, atol=2e-5)
    dfa.close()


# ---------------------------------------------------------------- decode loop on the head step
@pytest.mark.parametrize("kind,V,H,B,steps", [("dfa", 3000, 128, 300, 8), ("trie", 2000, 192, 150, 5),
                                              ("dfa", 700, 64, 1, 4)])
def test_head_decode_loop_exact_inputs(cd, oracle, mode, kind, V, H, B, steps):
    """cd_head_decode_loop against O7 on exact-arithmetic inputs: bit-exact histories, lengths,
    final states and done flags; sum of log-probs within the sum of the per-step bounds."""
    if kind == "dfa":
        aut = wl.make_random_dfa(23, V, 20, 0.1, 0.15)
    else:
        aut = wl.make_trie(V, wl.draw_labels(23, V, 25, 1, 5))
    dfa = dev_dfa(cd, aut, mode)
    W = wl.make_head(23, V, H, 2.0, exact=True)
    hs = [wl.make_hidden(23, k, B, H, exact=True) for k in range(steps)]
    got = cd.head_decode_loop(dfa, [h.to("cuda:0") for h in hs], W.to("cuda:0"), H=H)
    torch.cuda.synchronize()
    want = oracle.head_decode_loop(aut, hs, W, H)
    for k in ("tokens", "len", "final_state", "done"):
        assert np.array_equal(got[k].cpu().numpy(), want[k]), k
    slp = got["sum_logprob"].cpu().numpy().astype(np.float64)
    bound = TOL * (want["len"] + np.abs(want["sum_logprob"]))
    assert np.all(np.abs(slp - want["sum_logprob"]) <= bound + 1e-12)
    assert want["len"].max() > 1 or B == 1


def test_head_decode_loop_matches_logits_loop(cd, mode):
    """Same loop through cd_decode_loop on fp32 logits formed by a library matmul (exact inputs):
    the two entry points of the library agree bit for bit."""
    V, H, B, steps = 4096, 256, 200, 6
    aut = wl.make_random_dfa(29, V, 30, 0.05, 0.1)
    dfa = dev_dfa(cd, aut, mode)
    W = wl.make_head(29, V, H, 2.0, exact=True, device="cuda:0")
    hs = [wl.make_hidden(29, k, B, H, exact=True, device="cuda:0") for k in range(steps)]
    logits = [(h.float() @ W.float().t()).contiguous() for h in hs]  # exact in fp32
    a = cd.head_decode_loop(dfa, hs, W, H=H)
    b = cd.decode_loop(dfa, logits)
    torch.cuda.synchronize()
    for k in ("tokens", "len", "final_state", "done"):
        assert torch.equal(a[k], b[k]), k


def test_head_decode_loop_host_equals_device_loop(cd, mode):
    """cd_head_decode_loop_host (pinned host hidden states in, host outputs) against the device-buffer loop."""
    V, H, B, steps = 4096, 256, 200, 6
    aut = wl.make_random_dfa(29, V, 30, 0.05, 0.1)
    dfa = dev_dfa(cd, aut, mode)
    W = wl.make_head(29, V, H, 2.0, device="cuda:0")
    hs = [wl.make_hidden(29, k, B, H) for k in range(steps)]
    pinned = [h.pin_memory() for h in hs]
    a = cd.head_decode_loop_host(dfa, pinned, W, H=H)
    b = cd.head_decode_loop(dfa, [h.to("cuda:0") for h in hs], W, H=H)
    torch.cuda.synchronize()
    for k in ("tokens", "len", "final_state", "done", "sum_logprob"):
        assert torch.equal(a[k], b[k].cpu()), k
    assert not a["tokens"].is_cuda and int(a["len"].max()) > 1


# ---------------------------------------------------------------- sampling on the head path (N5 x N2)
@pytest.mark.parametrize("V,H,S,n,density,T", [(3000, 128, 12, 150, 0.1, 1.0), (5000, 256, 8, 300, 1.0, 0.6),
                                               (1000, 200, 7, 37, 0.3, 2.0)])
def test_head_sampled_step_matches_oracle_on_exact_logits(cd, oracle, mode, V, H, S, n, density, T):
    """cd_set_sampling on cd_head_step against O10 applied to fp32 logits from a library matmul
    (exact-arithmetic inputs: the head's fp32 dot products equal them bit for bit)."""
    aut = wl.make_random_dfa(71, V, S, density, 0.2)
    dfa = dev_dfa(cd, aut, mode)
    dfa.set_sampling(T, seed=0xABCDEF0123, step_base=3)
    hid = wl.make_hidden(71, 0, n + 9, H, exact=True)
    W = wl.make_head(71, V, H, 2.0, exact=True)
    x32 = (hid.double() @ W.double().t()).float().contiguous()
    states = live_states(aut, n)
    row_map = [(i * 5 + 2) % (n + 9) for i in range(n)]
    st_d = torch.tensor(states, dtype=torch.int32, device="cuda:0")
    rm_d = torch.tensor(row_map, dtype=torch.int32, device="cuda:0")
    tok, lp, lse, done = cd.head_step(dfa, hid.to("cuda:0"), W.to("cuda:0"), st_d, row_map=rm_d, H=H)
    torch.cuda.synchronize()
    o_tok, o_lp, o_lse, o_done, o_st = oracle.sample_step(aut, x32, states, T, seed=0xABCDEF0123, step=3, row_map=row_map)
    assert tok.cpu().numpy().tolist() == o_tok.tolist()
    assert st_d.cpu().numpy().tolist() == o_st.tolist() and done.cpu().numpy().tolist() == o_done.tolist()
    for g, r in ((lp, o_lp), (lse, o_lse)):
        assert np.all(np.abs(g.cpu().numpy().astype(np.float64) - r) <= TOL * np.maximum(1.0, np.abs(r)))


def test_head_sampled_loop_matches_logits_loop(cd, oracle, mode):
    V, H, B, steps = 4096, 256, 200, 6
    aut = wl.make_random_dfa(73, V, 30, 0.05, 0.1)
    dfa = dev_dfa(cd, aut, mode)
    dfa.set_sampling(0.8, seed=17, step_base=1)
    W = wl.make_head(73, V, H, 2.0, exact=True)
    hs = [wl.make_hidden(73, k, B, H, exact=True) for k in range(steps)]
    logits = [(h.double() @ W.double().t()).float().contiguous() for h in hs]
    got = cd.head_decode_loop(dfa, [h.to("cuda:0") for h in hs], W.to("cuda:0"), H=H)
    torch.cuda.synchronize()
    want = oracle.sample_decode_loop(aut, logits, 0.8, seed=17, step_base=1)
    for k in ("tokens", "len", "final_state", "done"):
        assert np.array_equal(got[k].cpu().numpy(), want[k]), k
    slp = got["sum_logprob"].cpu().numpy().astype(np.float64)
    assert np.all(np.abs(slp - want["sum_logprob"]) <= TOL * (want["len"] + np.abs(want["sum_logprob"])) + 1e-12)


def test_head_loop_many_rows(cd, oracle, mode):
    """B = 6,000 rows (47 row tiles, more than one chunk of the one-CTA list building) on the head path."""
    V, H, B, steps = 1536, 64, 6000, 4
    aut = wl.make_random_dfa(79, V, 16, 0.08, 0.2)
    dfa = dev_dfa(cd, aut, mode)
    W = wl.make_head(79, V, H, 2.0, exact=True)
    hs = [wl.make_hidden(79, k, B, H, exact=True) for k in range(steps)]
    got = cd.head_decode_loop(dfa, [h.to("cuda:0") for h in hs], W.to("cuda:0"), H=H)
    torch.cuda.synchronize()
    want = oracle.head_decode_loop(aut, hs, W, H)
    for k in ("tokens", "len", "final_state", "done"):
        assert np.array_equal(got[k].cpu().numpy(), want[k]), k
    assert want["n_active_hist"][1] > 4096


def test_head_step_changing_hidden_size_on_one_handle(cd, oracle):
    """One handle / stream used with H = 200, then H = 72, then H = 200 again (K tails in both): the packed
    A operand and its tensor map must follow H."""
    V, S, n = 900, 6, 70
    aut = wl.make_random_dfa(83, V, S, 0.3, 0.2)
    dfa = cd.compile_dfa(aut.V, aut.S, aut.start, aut.row_ptr, aut.tok, aut.next, aut.accepting, device="cuda:0")
    dfa.set_head_gather_max(0)
    for H in (200, 72, 200, 8):
        hid = wl.make_hidden(83 + H, 0, n, H, exact=True)
        W = wl.make_head(83 + H, V, H, 2.0, exact=True)
        run_case(cd, oracle, aut, dfa, hid, W, H, live_states(aut, n))
