"""Parity of the CUDA path (through the C ABI) with the CPU oracle, element by
element on the same seeded inputs.

Bar (BASELINE.json north_star): bit-exact token ids, next states, done flags
and compacted row order; log-probs / lse within 1e-5 relative with fp32
accumulation, read as abs(gpu - ref) <= 1e-5 * max(1, |ref|) (SURVEY 8(c) G9:
-log(sum) is ill-conditioned relative to itself near 0; DESIGN.md derives the
bound from the arithmetic).
"""
import math
import threading

import numpy as np
import pytest
import torch

import workloads as wl
from golden_util import read_decode

pytestmark = pytest.mark.gpu

TOL = 1e-5


@pytest.fixture(scope="module")
def cd():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    import paper_2606_31808_b200 as m

    m.lib()
    return m


# Every test of this module runs three times: dense scan only (the method as BASELINE.json
# north_star states it), every state gathered through its CSR token list, and a mix (states
# with at most the median number of transitions gathered) -- SURVEY 8(f) N1: same outputs, same
# oracle, same tolerances.
_MODE = {"name": "dense"}


@pytest.fixture(autouse=True, params=["dense", "gather_all", "gather_mixed"])
def step_mode(request):
    _MODE["name"] = request.param
    yield request.param
    _MODE["name"] = "dense"


def dev_dfa(cd, aut):
    dfa = cd.compile_dfa(aut.V, aut.S, aut.start, aut.row_ptr, aut.tok, aut.next, aut.accepting, device="cuda:0")
    return apply_mode(dfa, aut)


def apply_mode(dfa, aut):
    if _MODE["name"] == "gather_all":
        dfa.set_gather_max(2**30)
    elif _MODE["name"] == "gather_mixed":
        deg = torch.diff(torch.as_tensor(aut.row_ptr).cpu())
        deg = deg[deg > 0]
        dfa.set_gather_max(max(1, int(deg.median())) if deg.numel() else 1)
    return dfa


def close(gpu, ref, tol=TOL):
    gpu = np.asarray(gpu, np.float64)
    ref = np.asarray(ref, np.float64)
    both_inf = np.isneginf(gpu) & np.isneginf(ref)
    err = np.abs(np.where(both_inf, 0.0, gpu - ref))
    bound = tol * np.maximum(1.0, np.abs(np.where(both_inf, 0.0, ref)))
    return bool(np.all(err <= bound)), float(np.max(err / bound)) if err.size else 0.0


def check_step(cd, oracle, aut, dfa, x_dev, states, row_map=None):
    """One cd_step call against oracle.step on the same bytes."""
    st_dev = torch.tensor(states, dtype=torch.int32, device="cuda:0")
    rm_dev = None if row_map is None else torch.tensor(row_map, dtype=torch.int32, device="cuda:0")
    tok, lp, lse, done = cd.step(dfa, x_dev, st_dev, row_map=rm_dev)
    torch.cuda.synchronize()
    o_tok, o_lp, o_lse, o_done, o_st = oracle.step(aut, x_dev.cpu(), states, row_map=row_map)
    assert tok.cpu().numpy().tolist() == o_tok.tolist()
    assert st_dev.cpu().numpy().tolist() == o_st.tolist()
    assert done.cpu().numpy().tolist() == o_done.tolist()
    ok, worst = close(lp.cpu().numpy(), o_lp)
    assert ok, f"logprob off by {worst:.2f}x the bound"
    ok, worst = close(lse.cpu().numpy(), o_lse)
    assert ok, f"lse off by {worst:.2f}x the bound"
    return tok, lp, lse, done


def live_states(aut, n, stride=7):
    live = [s for s in range(aut.S) if not aut.accepting[s]]
    return [live[(stride * i) % len(live)] for i in range(n)]


# ------------------------------------------------------------------ the step
@pytest.mark.parametrize("dtype", [torch.float32, torch.bfloat16])
@pytest.mark.parametrize(
    "V,S,density,n",
    [
        (64, 5, 0.3, 9),          # one partial tile
        (37, 4, 0.3, 11),         # row bytes not a multiple of 16: scalar tail path
        (5001, 9, 0.03, 50),      # several tiles + 1-element tail after the bulk copy
        (1024, 8, 0.05, 33),      # exactly one fp32 tile
        (2048, 8, 0.05, 33),      # exactly one bf16 tile
        (5000, 12, 0.02, 70),     # several tiles + ragged tail, V % 32 != 0
        (40000, 16, 0.02, 301),   # many tiles, ragged
        (262144, 6, 0.005, 24),   # full vocabulary, few rows (row split over many units)
    ],
)
def test_step_matches_oracle_random_dfa(cd, oracle, dtype, V, S, density, n):
    aut = wl.make_random_dfa(seed=V + S, V=V, S=S, density=density, accept_frac=0.25, device="cuda:0")
    dfa = dev_dfa(cd, aut)
    ld = (V + 7) // 8 * 8
    x = wl.make_logits(V, 0, n, V, 2.0, dtype, device="cuda:0", ld=ld)
    states = live_states(aut, n)
    check_step(cd, oracle, aut, dfa, x, states)
    # mixed with already-accepted slots (never advance) and a row_map permutation
    acc = [s for s in range(S) if aut.accepting[s]]
    if acc:
        states2 = [acc[i % len(acc)] if i % 3 == 0 else s for i, s in enumerate(states)]
        perm = np.random.default_rng(n).permutation(n).astype(np.int32)
        check_step(cd, oracle, aut, dfa, x, states2, row_map=perm)
    dfa.close()


@pytest.mark.parametrize("dtype", [torch.float32, torch.bfloat16])
def test_step_dense_masks(cd, oracle, dtype):
    """All tokens allowed (reduces to textbook log-softmax/argmax) and 50 % density."""
    for V, density in ((4096, 1.0), (10000, 1.0), (10000, 0.5)):
        aut = wl.make_random_dfa(seed=17, V=V, S=3, density=density, accept_frac=0.0, device="cuda:0")
        dfa = dev_dfa(cd, aut)
        ld = (V + 7) // 8 * 8
        x = wl.make_logits(3, 0, 40, V, 3.0, dtype, device="cuda:0", ld=ld)
        states = [i % 3 for i in range(40)]
        tok, lp, lse, _ = check_step(cd, oracle, aut, dfa, x, states)
        if density == 1.0:  # independent library pin on the GPU result itself
            xd = x[:, :V].double()
            ref = torch.logsumexp(xd, dim=1)
            assert torch.allclose(lse.double(), ref, rtol=0, atol=1e-5 * float(ref.abs().max().clamp(min=1)))
            m = xd.max(dim=1).values
            first = torch.stack([torch.nonzero(xd[i] == m[i])[0, 0] for i in range(40)])
            assert tok.cpu().tolist() == first.cpu().tolist()
        dfa.close()


def _subset_aut(V, toks):
    toks = sorted(toks)
    return wl.Automaton(
        V=V, S=2, start=0,
        row_ptr=torch.tensor([0, len(toks), len(toks)], dtype=torch.int64),
        tok=torch.tensor(toks, dtype=torch.int32),
        next=torch.ones(len(toks), dtype=torch.int32),
        accepting=torch.tensor([0, 1], dtype=torch.uint8),
    )


@pytest.mark.parametrize("dtype", [torch.float32, torch.bfloat16])
def test_planted_ties_across_work_boundaries(cd, oracle, dtype):
    """Equal maxima at lane / word / tile / unit / row boundaries: lowest id wins."""
    V = 262144
    tile = 1024 if dtype == torch.float32 else 2048
    groups = [
        [31, 32], [63, 64, 65], [tile - 1, tile], [2 * tile - 1, 2 * tile, 2 * tile + 1],
        [16 * tile - 1, 16 * tile], [0, V - 1], [V // 2 - 1, V // 2, V - 1], [5, 100000, 200000, 262143],
        [tile * 7 + 31, tile * 8 + 0, tile * 9 + 33],
    ]
    n = len(groups) * 2
    g = torch.Generator(device="cuda:0").manual_seed(1)
    x = (torch.randn(n, V, generator=g, device="cuda:0") * 2.0).clamp_(max=5.0)
    for i, ids in enumerate(groups):
        x[2 * i, ids] = 6.0
        x[2 * i + 1, ids] = 6.0
    x = x.to(dtype)
    all_ones = _subset_aut(V, range(V))
    dfa = dev_dfa(cd, all_ones)
    tok, _, _, _ = check_step(cd, oracle, all_ones, dfa, x, [0] * n)
    assert tok.cpu().tolist() == [ids[0] for ids in groups for _ in (0, 1)]
    dfa.close()
    # the same with a sparse allowed set that drops the lowest planted id of each group
    allowed = set(range(0, V, 97))
    for ids in groups:
        allowed.update(ids[1:])
        allowed.discard(ids[0])
    sparse = _subset_aut(V, allowed)
    dfa = dev_dfa(cd, sparse)
    tok, _, _, _ = check_step(cd, oracle, sparse, dfa, x, [0] * n)
    assert tok.cpu().tolist() == [ids[1] for ids in groups for _ in (0, 1)]
    dfa.close()


def test_closed_forms_on_gpu(cd, oracle):
    V = 8192
    aut = _subset_aut(V, [9, 4100])
    dfa = dev_dfa(cd, aut)
    pairs = [(0.5, -1.25), (-3.0, -3.0), (10.0, 9.0), (-20.0, 1.0), (100.0, 80.0), (0.0, 0.0)]
    x = torch.full((len(pairs), V), 50.0, device="cuda:0")
    for i, (a, b) in enumerate(pairs):
        x[i, 9], x[i, 4100] = a, b
    tok, lp, lse, done = check_step(cd, oracle, aut, dfa, x, [0] * len(pairs))
    for i, (a, b) in enumerate(pairs):
        assert int(tok[i]) == (9 if a >= b else 4100)
        want = -math.log1p(math.exp(-abs(a - b)))
        assert abs(float(lp[i]) - want) <= TOL
    dfa.close()
    one = _subset_aut(V, [4000])
    dfa = dev_dfa(cd, one)
    x = torch.randn(5, V, device="cuda:0")
    tok, lp, lse, _ = check_step(cd, oracle, one, dfa, x, [0] * 5)
    assert tok.cpu().tolist() == [4000] * 5 and lp.cpu().tolist() == [0.0] * 5
    assert torch.equal(lse, x[:, 4000])
    dfa.close()


@pytest.mark.parametrize("dtype", [torch.float32, torch.bfloat16])
def test_special_values(cd, oracle, dtype):
    V = 4096
    ids = [4, 800, 1500, 4095]
    aut = _subset_aut(V, ids)
    dfa = dev_dfa(cd, aut)
    ninf, nan = -float("inf"), float("nan")
    rows = [
        [nan, 1.0, nan, 1.0],       # NaN read as -inf
        [ninf, ninf, ninf, ninf],   # all -inf: lowest allowed id, logprob = lse = -inf
        [nan, nan, nan, nan],       # all NaN: same
        [ninf, 2.0, 2.0, ninf],
        [-0.0, 0.0, -5.0, -5.0],    # signed zeros tie
        [3e38, 3e38, -3e38, 0.0],
    ]
    x = torch.zeros((len(rows), V), device="cuda:0")
    for i, r in enumerate(rows):
        x[i, ids] = torch.tensor(r, device="cuda:0")
    x = x.to(dtype)
    tok, lp, lse, _ = check_step(cd, oracle, aut, dfa, x, [0] * len(rows))
    assert tok.cpu().tolist()[:5] == [800, 4, 4, 800, 4]
    assert float(lp[1]) == ninf and float(lse[1]) == ninf
    # poisoned complement: disallowed logits must never matter
    base = [t.clone() for t in cd.step(dfa, x, torch.zeros(len(rows), dtype=torch.int32, device="cuda:0"))]
    for poison in (1e30, float("inf"), nan, ninf):
        y = x.clone().float()
        dis = torch.ones(V, dtype=torch.bool, device="cuda:0")
        dis[ids] = False
        y[:, dis] = poison
        out = cd.step(dfa, y.to(dtype), torch.zeros(len(rows), dtype=torch.int32, device="cuda:0"))
        for a, b in zip(base, out):
            assert torch.equal(a.view(torch.uint8) if a.dtype != torch.uint8 else a,
                               b.view(torch.uint8) if b.dtype != torch.uint8 else b)
    # +inf: only the token is defined (lowest +inf id); parity of the values is unpinned (G6)
    x2 = torch.zeros((1, V), device="cuda:0")
    x2[0, 1500] = x2[0, 800] = float("inf")
    tok2, _, _, _ = cd.step(dfa, x2.to(dtype), torch.zeros(1, dtype=torch.int32, device="cuda:0"))
    assert int(tok2[0]) == 800
    dfa.close()


def test_step_n_zero_and_argument_errors(cd):
    aut = _subset_aut(64, [1, 2])
    dfa = dev_dfa(cd, aut)
    x = torch.zeros((4, 64), device="cuda:0")
    st = torch.zeros(0, dtype=torch.int32, device="cuda:0")
    tok, lp, lse, done = cd.step(dfa, x, st)
    assert tok.numel() == 0
    with pytest.raises(cd.CdError) as e:  # ld < V
        cd.step(dfa, torch.zeros((4, 32), device="cuda:0"), torch.zeros(4, dtype=torch.int32, device="cuda:0"))
    assert e.value.code == 1
    with pytest.raises(cd.CdError) as e:  # row stride not a multiple of 16 bytes
        cd.step(dfa, torch.zeros((4, 66), device="cuda:0"), torch.zeros(4, dtype=torch.int32, device="cuda:0"))
    assert e.value.code == 1
    with pytest.raises(cd.CdError) as e:  # misaligned base
        base = torch.zeros(4 * 64 + 4, device="cuda:0")
        cd.step(dfa, base[1:1 + 4 * 64].view(4, 64), torch.zeros(4, dtype=torch.int32, device="cuda:0"))
    assert e.value.code == 1
    dfa.close()


# ------------------------------------------------------------------ transition kernel
def test_transition_kernel(cd, oracle):
    aut = wl.make_random_dfa(seed=5, V=50000, S=40, density=0.02, accept_frac=0.2, device="cuda:0")
    dfa = dev_dfa(cd, aut)
    rng = np.random.default_rng(0)
    n = 3000
    states = rng.integers(0, aut.S, size=n).astype(np.int32)
    tokens = np.empty(n, np.int32)
    want_state = np.empty(n, np.int32)
    rp, tk, nx = aut.row_ptr.numpy(), aut.tok.numpy(), aut.next.numpy()
    for i, s in enumerate(states):
        lo, hi = rp[s], rp[s + 1]
        if i % 5 == 0 or hi == lo:  # token without a transition (or negative): state kept
            tokens[i] = -1 if i % 10 == 0 else int(rng.integers(0, aut.V))
            j = lo + np.searchsorted(tk[lo:hi], tokens[i])
            want_state[i] = nx[j] if (tokens[i] >= 0 and j < hi and tk[j] == tokens[i]) else s
        else:
            j = int(rng.integers(lo, hi))
            tokens[i], want_state[i] = tk[j], nx[j]
    st = torch.tensor(states, device="cuda:0")
    done = cd.transition(dfa, torch.tensor(tokens, device="cuda:0"), st)
    assert st.cpu().numpy().tolist() == want_state.tolist()
    assert done.cpu().numpy().tolist() == aut.accepting.numpy()[want_state].tolist()
    dfa.close()


# ------------------------------------------------------------------ compaction
@pytest.mark.parametrize("n", [0, 1, 2, 31, 32, 33, 1000, 1023, 1024, 1025, 4096, 4097, 70000])
@pytest.mark.parametrize("pattern", ["none", "all", "alt", "rand"])
def test_compaction_bit_exact(cd, oracle, n, pattern):
    rng = np.random.default_rng(n + 1)
    done = {
        "none": np.zeros(n, np.uint8),
        "all": np.ones(n, np.uint8),
        "alt": (np.arange(n) % 2).astype(np.uint8),
        "rand": (rng.random(n) < 0.3).astype(np.uint8),
    }[pattern]
    ids = np.sort(rng.choice(10 * n + 1, size=n, replace=False)).astype(np.int32)
    st = rng.integers(0, 5000, size=n).astype(np.int32)
    d = torch.tensor(done, device="cuda:0")
    ro, so, na = cd.compact(d, torch.tensor(ids, device="cuda:0"), torch.tensor(st, device="cuda:0"))
    o_ro, o_so, k = oracle.compact(done, ids, st)
    assert int(na) == k
    assert ro[:k].cpu().numpy().tolist() == o_ro.tolist()
    assert so[:k].cpu().numpy().tolist() == o_so.tolist()
    ro2, _, na2 = cd.compact(d)  # implicit ids
    assert int(na2) == k and ro2[:k].cpu().numpy().tolist() == [i for i in range(n) if not done[i]]


# ------------------------------------------------------------------ the loop
def check_loop(cd, oracle, aut, logits_dev, max_steps, ref=None, rows=None):
    """cd_decode_loop against O4, in all three loop modes: one launch per decoding step, the lock-step
    persistent kernel (grid barrier, bitmap-select instead of compaction) and the barrier-free persistent
    kernel (row groups advancing independently; the default).  Tokens, lengths, states and done flags
    must agree bit for bit; the first two also agree in the bits of the fp32 sums (same unit split, same
    merge order), the third splits rows into units per group, so its sums may differ in the last bits."""
    dfa = dev_dfa(cd, aut)
    dfa.set_loop_mode(cd.LOOP_PER_STEP)
    per_step = cd.decode_loop(dfa, logits_dev, max_steps=max_steps)
    assert dfa.loop_trace() == ([], [])
    dfa.set_loop_mode(cd.LOOP_BARRIER)
    lock = cd.decode_loop(dfa, logits_dev, max_steps=max_steps)
    for k in per_step:
        assert torch.equal(per_step[k].view(torch.uint8) if per_step[k].dtype == torch.float32 else per_step[k],
                           lock[k].view(torch.uint8) if lock[k].dtype == torch.float32 else lock[k]), ("loop modes differ", k)
    dfa.set_loop_mode(cd.LOOP_AUTO)
    out = cd.decode_loop(dfa, logits_dev, max_steps=max_steps)
    for k in ("tokens", "len", "final_state", "done"):
        assert torch.equal(lock[k], out[k]), ("loop modes differ", k)
    fin = torch.isfinite(lock["sum_logprob"])
    assert torch.equal(fin, torch.isfinite(out["sum_logprob"]))
    assert torch.all((lock["sum_logprob"][fin] - out["sum_logprob"][fin]).abs() <=
                     1e-5 * (out["len"][fin] + out["sum_logprob"][fin].abs()).clamp(min=1))
    if ref is None:
        ref = oracle.decode_loop(aut, [x.cpu() for x in logits_dev], max_steps=max_steps)
    B = logits_dev[0].shape[0]
    if B <= 32768 and not bool(aut.accepting[aut.start]) and rows is None and "n_active_hist" in ref:
        # the persistent kernel ran, and its per-step active counts are the oracle's
        n_tr, t_tr = dfa.loop_trace()
        hist = [int(v) for v in ref["n_active_hist"] if v > 0]
        assert n_tr == hist, (n_tr, hist)
        assert all(t >= 0 for t in t_tr) and sum(t_tr) > 0
    sel = slice(None) if rows is None else rows
    for k in ("tokens", "len", "final_state", "done"):
        assert np.array_equal(out[k].cpu().numpy()[sel], ref[k]), k
    g, r = out["sum_logprob"].cpu().numpy().astype(np.float64)[sel], ref["sum_logprob"]
    bound = TOL * (ref["len"] + np.abs(np.where(np.isinf(r), 0, r)))  # sum of per-step bounds
    fin = np.isfinite(r)
    assert np.array_equal(np.isfinite(g), fin)
    assert np.all(np.abs(g[fin] - r[fin]) <= np.maximum(bound[fin], TOL)), float(np.max(np.abs(g[fin] - r[fin])))
    dfa.close()
    return out, ref


def test_loop_c0_against_golden(cd, oracle):
    """BASELINE.json configs[0] exactly as stated; expectation is the stored oracle result."""
    cfg = wl.CONFIGS["c0"]
    aut = wl.build_automaton(cfg)
    logits = wl.build_step_logits(cfg, aut, device="cpu")  # the fixture was made from CPU-generated logits
    gold = read_decode("c0_decode.txt")
    out, _ = check_loop(cd, oracle, aut, [x.cuda() for x in logits], cfg.max_steps, ref=gold)
    labels = {(17, 3), (42,)}
    for r in range(cfg.B):
        assert tuple(out["tokens"][r, : int(out["len"][r])].cpu().tolist()) in labels


def test_loop_c3_small_against_golden(cd, oracle):
    cfg = wl.scaled(wl.CONFIGS["c3"], V=4096, B=48, S=64, max_steps=10)
    aut = wl.build_automaton(cfg)
    logits = wl.build_step_logits(cfg, aut, device="cpu")
    check_loop(cd, oracle, aut, [x.cuda() for x in logits], cfg.max_steps, ref=read_decode("c3_small_decode.txt"))


def test_async_loops_back_to_back(cd, oracle):
    """cd_decode_loop_async: three loops enqueued back to back on one stream (one kernel launch each, shared
    scratch), one cd_loop_sync; every one matches the oracle, and the synchronous call bit for bit."""
    cfg = wl.scaled(wl.CONFIGS["c3"], V=8192, B=300, S=64, max_steps=9)
    aut = wl.build_automaton(cfg)
    dfa = dev_dfa(cd, aut)
    batches = [wl.build_step_logits(cfg, aut, device="cuda:0", batch=i) for i in range(3)]
    preps = [cd.PreparedLoop(dfa, b) for b in batches]
    n0 = cd.launch_count()
    for p in preps:
        p.enqueue()
    launched = cd.launch_count() - n0
    preps[0].sync()
    assert launched == 3, launched
    for p, b in zip(preps, batches):
        ref = oracle.decode_loop(aut, [x.cpu() for x in b], max_steps=cfg.max_steps)
        for k in ("tokens", "len", "final_state", "done"):
            assert np.array_equal(p.out[k].cpu().numpy(), ref[k]), k
        sync_out = cd.decode_loop(dfa, b)
        for k in ("tokens", "len", "final_state", "done", "sum_logprob"):
            assert torch.equal(sync_out[k], p.out[k]), k
        g, r = p.out["sum_logprob"].cpu().numpy().astype(np.float64), ref["sum_logprob"]
        fin = np.isfinite(r)
        assert np.array_equal(np.isfinite(g), fin)
        assert np.all(np.abs(g[fin] - r[fin]) <= np.maximum(TOL * (ref["len"] + np.abs(r))[fin], TOL))
    # the per-step path enqueues too (LIMIT-free loops in CD_LOOP_PER_STEP mode)
    dfa.set_loop_mode(cd.LOOP_PER_STEP)
    q = cd.PreparedLoop(dfa, batches[1])
    q.enqueue()
    q.sync()
    for k in ("tokens", "len", "final_state", "done"):
        assert torch.equal(q.out[k], preps[1].out[k]), k
    dfa.close()


def test_loop_accepting_start(cd, oracle):
    aut = wl.Automaton(V=64, S=1, start=0, row_ptr=torch.tensor([0, 1]), tok=torch.tensor([1], dtype=torch.int32),
                       next=torch.tensor([0], dtype=torch.int32), accepting=torch.tensor([1], dtype=torch.uint8))
    check_loop(cd, oracle, aut, [torch.zeros(5, 64, device="cuda:0")] * 3, 3)


@pytest.mark.parametrize("name", ["c1", "c2", "c3"])
def test_loop_full_size_configs(cd, oracle, name):
    """BASELINE.json configs[1..3] at full size, element by element (the oracle
    only touches allowed logits, so it finishes in seconds even at V=262144)."""
    cfg = wl.CONFIGS[name]
    aut = wl.build_automaton(cfg, device="cuda:0")
    assert oracle.validate(aut) == 0
    logits = wl.build_step_logits(cfg, aut, device="cuda:0")
    out, ref = check_loop(cd, oracle, aut, logits, cfg.max_steps)
    if aut.labels is not None:  # tries: every decoded history is one of the labels
        leaf = {tuple(l): aut.leaf_of_label[i] for i, l in enumerate(aut.labels)}
        toks, ln, fs = out["tokens"].cpu().numpy(), out["len"].cpu().numpy(), out["final_state"].cpu().numpy()
        for r in range(cfg.B):
            h = tuple(toks[r, : ln[r]].tolist())
            assert h in leaf and fs[r] == leaf[h]
        assert bool(out["done"].all())
    else:  # statistics sanity: survival ~ (1 - accept_frac)^k
        acc = float(aut.accepting.float().mean())
        hist = ref["n_active_hist"]
        for k in range(0, cfg.max_steps, 4):
            expect = cfg.B * (1 - acc) ** k
            assert abs(hist[k] - expect) < 6 * math.sqrt(cfg.B) + 0.15 * expect


def test_step_and_loop_are_bitwise_reproducible(cd, oracle, step_mode):
    """Stand-in for racecheck (compute-sanitizer is closed on this pool): the fence-free, ticket-free
    merge of the unit results (cd_step.cuh: tagged 64-bit slots polled by the warp that holds a row's
    last part) and the grid barrier / bitmap rotation of the persistent loop must give IDENTICAL BITS on
    every run.  The same c4-shaped cd_step and cd_decode_loop are run 200 times at n in {8, 148, 1024,
    4096}, on two streams at once (two grids sharing the SMs: the merge waits only for units that were
    drawn earlier, so partial residency must not deadlock it), and compared with the first run."""
    cfg = wl.CONFIGS["c4"]
    free, _ = torch.cuda.mem_get_info()
    if free < 12 * 2**30:
        pytest.skip("needs ~10 GiB of device memory")
    aut = wl.build_automaton(cfg, device="cuda:0")
    dfa = dev_dfa(cd, aut)
    xs = [wl.make_logits(cfg.seed, k, cfg.B, cfg.V, cfg.std, cfg.dtype, device="cuda:0") for k in range(2)]
    live = live_states(aut, cfg.B)
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    reps = 200
    for n in (8, 148, 1024, 4096):
        st0 = torch.tensor(live[:n], dtype=torch.int32, device="cuda:0")
        steps = [xs[k & 1][:n] for k in range(cfg.max_steps)]
        first_step, first_loop = None, {}
        torch.cuda.synchronize()
        for rep in range(0, reps, 2):
            got = []
            for si, stream in enumerate(streams):
                with torch.cuda.stream(stream):
                    st = st0.clone()
                    tok, lp, lse, done = cd.step(dfa, xs[0], st, n=n)
                    got.append((tok, lp, lse, done, st))
            # the loops synchronise their stream before returning: two host threads keep both streams busy
            loops = [None, None]

            def run_loop(si):
                with torch.cuda.stream(streams[si]):
                    loops[si] = cd.decode_loop(dfa, steps)

            # the bits must repeat (since the canonical chunk arithmetic the three kernels also agree with one another:
            # test_results_do_not_depend_on_the_batch)
            lmode = (cd.LOOP_AUTO, cd.LOOP_BARRIER, cd.LOOP_PER_STEP)[(rep // 2) % 3]
            dfa.set_loop_mode(lmode)
            threads = [threading.Thread(target=run_loop, args=(si,)) for si in range(2)]
            for t in threads:
                t.start()
            for t in threads:
                t.join()
            torch.cuda.synchronize()
            for g in got:
                cur = [t.view(torch.uint8) if t.dtype == torch.float32 else t for t in g]
                if first_step is None:
                    first_step = [t.clone() for t in cur]
                for a, b in zip(first_step, cur):
                    assert torch.equal(a, b), ("cd_step not reproducible", n, rep)
            for lo in loops:
                cur = {k: (v.view(torch.uint8) if v.dtype == torch.float32 else v) for k, v in lo.items()}
                if lmode not in first_loop:
                    first_loop[lmode] = {k: v.clone() for k, v in cur.items()}
                for k in cur:
                    assert torch.equal(first_loop[lmode][k], cur[k]), ("cd_decode_loop not reproducible", n, rep, lmode, k)
        # and the first run is right (8 and 148 rows: the oracle in full; larger n: the first 256 rows)
        m = min(n, 256)
        o_tok, o_lp, o_lse, o_done, o_st = oracle.step(aut, xs[0][:m].cpu(), live[:m])
        assert first_step[0][:m].cpu().numpy().tolist() == o_tok.tolist()
        assert first_step[4][:m].cpu().numpy().tolist() == o_st.tolist()
        want = oracle.decode_loop(aut, [x[:m].cpu() for x in steps])
        for lmode in first_loop:
            assert np.array_equal(first_loop[lmode]["tokens"][:m].cpu().numpy(), want["tokens"]), lmode
    dfa.set_loop_mode(cd.LOOP_AUTO)
    dfa.close()


def test_results_do_not_depend_on_the_batch(cd, oracle, step_mode):
    """The canonical arithmetic of cd_step.cuh: a row is cut into chunks that depend on V and the logits type only,
    a chunk's result is a fixed function of its elements and a row's result a fixed fold of its chunks' -- so how a
    launch cuts rows into units (which depends on the number of active rows, on the kernel and, in the row-task loop,
    on how busy the machine is) must not change a BIT of logprob / lse.  The same rows are decoded alone, in small and
    large batches, permuted, through cd_step and through the three loop kernels."""
    cfg = wl.scaled(wl.CONFIGS["c4"], B=1500, S=256, max_steps=6)
    aut = wl.build_automaton(cfg, device="cuda:0")
    dfa = dev_dfa(cd, aut)
    xs = wl.build_step_logits(cfg, aut, device="cuda:0")
    live = live_states(aut, cfg.B)

    def bits(t):
        return t.view(torch.int32) if t.dtype == torch.float32 else t

    # cd_step: all rows at once is the reference
    st = torch.tensor(live, dtype=torch.int32, device="cuda:0")
    tok0, lp0, lse0, done0 = cd.step(dfa, xs[0], st)
    st0 = st.clone()
    g = torch.Generator().manual_seed(5)
    for n in (1, 2, 37, 148, 1024):
        rows = torch.randperm(cfg.B, generator=g)[:n].to("cuda:0")
        rm = rows.to(torch.int32)
        st = torch.tensor(live, dtype=torch.int32, device="cuda:0")[rows].contiguous()
        tok, lp, lse, done = cd.step(dfa, xs[0], st, row_map=rm)
        assert torch.equal(tok, tok0[rows]) and torch.equal(st, st0[rows]) and torch.equal(done, done0[rows])
        assert torch.equal(bits(lp), bits(lp0[rows])), ("logprob bits depend on the batch", n)
        assert torch.equal(bits(lse), bits(lse0[rows])), ("lse bits depend on the batch", n)
    # the loops: three kernels, whole batch and sub-batches
    ref = None
    for lmode in (cd.LOOP_AUTO, cd.LOOP_BARRIER, cd.LOOP_PER_STEP):
        dfa.set_loop_mode(lmode)
        for B in (cfg.B, 700, 3):
            out = cd.decode_loop(dfa, [x[:B] for x in xs])
            cur = {k: bits(v).clone() for k, v in out.items()}
            if ref is None:
                ref = cur
            for k in cur:
                assert torch.equal(cur[k], ref[k][:B]), ("loop results depend on the kernel or the batch", lmode, B, k)
    dfa.set_loop_mode(cd.LOOP_AUTO)
    # ... and the common result is the oracle's
    want = oracle.decode_loop(aut, [x.cpu() for x in xs])
    assert np.array_equal(ref["tokens"].cpu().numpy(), want["tokens"])
    dfa.close()


@pytest.mark.parametrize("V,B,steps,S", [(262144, 8, 300, 64), (2048, 3000, 300, 48)])
def test_long_loops_wrap_the_queue_ring(cd, oracle, V, B, steps, S):
    """Loops far longer than anything the configs need: more steps than fit the kernel's parameter block (the step
    pointers then live in device memory), more than the 256 steps the device-side trace records, and more queue
    entries than the ring of the row-task kernel holds -- a few rows cut into 64 units per step (V = 262144), or
    thousands of rows of one unit each (V = 2048) -- so the ring wraps several times and its tags (launch generation +
    wrap count) are what tells a fresh entry from the one a slot held before.  Almost no state accepts, so most rows
    run to max_steps.  All three loop kernels against the oracle."""
    aut = wl.make_random_dfa(91, V, S, 0.01 if V > 4096 else 0.05, 0.004)
    dfa = dev_dfa(cd, aut)
    nbuf = 7  # the steps cycle through 7 logits buffers (the API takes one pointer per step)
    bufs = [wl.make_logits(91, k, B, V, 2.0, torch.bfloat16, device="cuda:0") for k in range(nbuf)]
    xs = [bufs[k % nbuf] for k in range(steps)]
    want = oracle.decode_loop(aut, [x.cpu() for x in bufs] * (steps // nbuf + 1), max_steps=steps)
    assert int((want["len"] == steps).sum()) > B // 4  # long-lived rows: the loop really is long
    for lm in (cd.LOOP_AUTO, cd.LOOP_BARRIER, cd.LOOP_PER_STEP):
        dfa.set_loop_mode(lm)
        for rep in range(2):  # twice: the second launch finds the ring full of the first one's entries
            out = cd.decode_loop(dfa, xs, max_steps=steps)
            for k in ("tokens", "len", "final_state", "done"):
                assert np.array_equal(out[k].cpu().numpy(), want[k]), (lm, rep, k)
            slp = out["sum_logprob"].cpu().numpy().astype(np.float64)
            assert np.all(np.abs(slp - want["sum_logprob"]) <= TOL * (want["len"] + np.abs(want["sum_logprob"])))
    dfa.set_loop_mode(cd.LOOP_AUTO)
    dfa.close()


@pytest.mark.parametrize("B", [1, 2, 32768, 32769, 50000])
def test_loop_row_count_boundaries(cd, oracle, B):
    """One row, two rows, the most rows a persistent loop kernel takes (32768), one more and many more (those run one
    launch per decoding step): the same results from whichever kernel the library picks, in every loop mode."""
    cfg = wl.scaled(wl.CONFIGS["c3"], V=1024, B=B, S=16, max_steps=4, density=0.06, dtype=torch.float32)
    aut = wl.build_automaton(cfg)
    dfa = dev_dfa(cd, aut)
    logits = wl.build_step_logits(cfg, aut, device="cuda:0")
    want = oracle.decode_loop(aut, [x.cpu() for x in logits])
    for lm in (cd.LOOP_AUTO, cd.LOOP_BARRIER, cd.LOOP_PER_STEP):
        dfa.set_loop_mode(lm)
        got = cd.decode_loop(dfa, logits)
        for k in ("tokens", "len", "final_state", "done"):
            assert np.array_equal(got[k].cpu().numpy(), want[k]), (lm, k)
        ok, worst = close(got["sum_logprob"].cpu().numpy(), want["sum_logprob"], tol=TOL * cfg.max_steps)
        assert ok, (lm, worst)
    dfa.set_loop_mode(cd.LOOP_AUTO)
    dfa.close()


def test_bad_state_is_reported_through_the_outputs_and_does_not_stick(cd, oracle):
    """A slot whose state is outside [0, S): cd_step cannot fail asynchronously, it reports the slot as
    done with token -1 and keeps the state; the error counter of the scratch area must not leak into the
    NEXT loop on the stream, which is clean and must return CD_OK (round-1 advice)."""
    cfg = wl.scaled(wl.CONFIGS["c3"], V=20000, B=64, S=32, max_steps=4)
    aut = wl.build_automaton(cfg)
    dfa = dev_dfa(cd, aut)
    logits = wl.build_step_logits(cfg, aut, device="cuda:0")
    live = live_states(aut, cfg.B)
    states = list(live)
    states[3], states[17], states[40] = aut.S, -1, aut.S + 1000
    st = torch.tensor(states, dtype=torch.int32, device="cuda:0")
    tok, lp, lse, done = cd.step(dfa, logits[0], st)
    torch.cuda.synchronize()
    good = [i for i in range(cfg.B) if i not in (3, 17, 40)]
    o_tok, o_lp, o_lse, o_done, o_st = oracle.step(aut, logits[0].cpu(), [states[i] for i in good], row_map=good)
    assert tok.cpu().numpy()[good].tolist() == o_tok.tolist() and st.cpu().numpy()[good].tolist() == o_st.tolist()
    for i in (3, 17, 40):
        assert int(tok[i]) == -1 and int(done[i]) == 1 and int(st[i]) == states[i] and float(lp[i]) == 0.0
    for lm in (cd.LOOP_AUTO, cd.LOOP_BARRIER, cd.LOOP_PER_STEP):  # the following loops are clean: CD_OK, right results
        dfa.set_loop_mode(lm)
        out = cd.decode_loop(dfa, logits)
        want = oracle.decode_loop(aut, [x.cpu() for x in logits])
        assert np.array_equal(out["tokens"].cpu().numpy(), want["tokens"])
    dfa.close()


@pytest.mark.parametrize("B", [37, 900])
def test_loop_states_of_very_different_degree(cd, oracle, B):
    """States with 1 ... 9000 transitions in one automaton: in the gather modes rows are split
    into different numbers of units per state, some units are drawn in vain, and a row's next
    state usually has another degree than the one it was processed in."""
    V, S, steps = 65536, 48, 14
    rng = np.random.default_rng(99)
    degs = [1, 2, 40, 255, 256, 257, 700, 1300, 2049, 5000, 9000, 3]
    row_ptr, tok, nxt = [0], [], []
    accepting = np.zeros(S, np.uint8)
    accepting[S - 3:] = 1
    for s in range(S):
        if accepting[s]:
            row_ptr.append(len(tok))
            continue
        d = degs[s % len(degs)]
        t = np.sort(rng.choice(V, size=d, replace=False))
        tok.extend(t.tolist())
        nxt.extend(rng.integers(0, S, size=d).tolist())
        row_ptr.append(len(tok))
    aut = wl.Automaton(V=V, S=S, start=0, row_ptr=torch.tensor(row_ptr, dtype=torch.int64),
                       tok=torch.tensor(tok, dtype=torch.int32), next=torch.tensor(nxt, dtype=torch.int32),
                       accepting=torch.tensor(accepting))
    assert oracle.validate(aut) == 0
    logits = [wl.make_logits(7, k, B, V, 2.0, torch.bfloat16, device="cuda:0") for k in range(steps)]
    check_loop(cd, oracle, aut, logits, steps)
    # and single steps from scattered states
    dfa = dev_dfa(cd, aut)
    states = [int(x) for x in rng.integers(0, S - 3, size=B)]
    check_step(cd, oracle, aut, dfa, logits[0], states)
    dfa.close()


# ------------------------------------------------------------------ LIMIT early exit
def check_limit_loop(cd, oracle, aut, dfa, logits, max_steps, sat, limit, counter):
    before = int(counter)
    out = cd.decode_loop(dfa, logits, max_steps=max_steps, limit=limit, satisfied=counter)
    ref = oracle.decode_loop(aut, [x.cpu() for x in logits], max_steps=max_steps, satisfying=sat, limit=limit,
                             satisfied=before)
    for k in ("tokens", "len", "final_state", "done"):
        assert np.array_equal(out[k].cpu().numpy(), ref[k]), k
    assert int(counter) == ref["satisfied"]
    g, r = out["sum_logprob"].cpu().numpy().astype(np.float64), ref["sum_logprob"]
    assert np.all(np.abs(g - r) <= np.maximum(TOL * (ref["len"] + np.abs(r)), TOL))
    return out, ref


@pytest.mark.parametrize("limit", [0, 1, 9, 60, 10**6])
def test_limit_early_exit_random_dfa(cd, oracle, limit):
    cfg = wl.scaled(wl.CONFIGS["c3"], V=40000, B=500, S=96, max_steps=12)
    aut = wl.build_automaton(cfg, device="cuda:0")
    logits = wl.build_step_logits(cfg, aut, device="cuda:0")
    acc = aut.accepting.cpu().numpy()
    sat = (acc * (np.arange(aut.S) % 2 == 0)).astype(np.uint8)
    dfa = dev_dfa(cd, aut)
    dfa.set_satisfying(sat)
    counter = torch.zeros(1, dtype=torch.int32, device="cuda:0")
    out, ref = check_limit_loop(cd, oracle, aut, dfa, logits, cfg.max_steps, sat, limit, counter)
    if limit == 10**6:  # never reached: identical to the plain loop
        plain = cd.decode_loop(dfa, logits, max_steps=cfg.max_steps)
        for k in plain:
            assert torch.equal(plain[k], out[k])
    if limit == 0:
        assert int(out["len"].max()) == 0 and int(counter) == 0
    # a second batch of the same query continues from the counter (usually: nothing runs)
    logits2 = wl.build_step_logits(cfg, aut, device="cuda:0", batch=1)
    check_limit_loop(cd, oracle, aut, dfa, logits2, cfg.max_steps, sat, limit, counter)
    dfa.close()


def test_limit_early_exit_boolean_filter_c1(cd, oracle):
    """`LLMMap(...) = TRUE ... LIMIT 10` on BASELINE.json configs[1] at full size."""
    cfg = wl.CONFIGS["c1"]
    aut = wl.build_automaton(cfg, device="cuda:0")
    logits = wl.build_step_logits(cfg, aut, device="cuda:0")
    sat = np.zeros(aut.S, np.uint8)
    sat[int(aut.leaf_of_label[0])] = 1
    dfa = dev_dfa(cd, aut)
    dfa.set_satisfying(sat)
    counter = torch.zeros(1, dtype=torch.int32, device="cuda:0")
    check_limit_loop(cd, oracle, aut, dfa, logits, cfg.max_steps, sat, 10, counter)
    dfa.close()


def test_limit_argument_errors(cd):
    aut = _subset_aut(64, [1, 2])
    dfa = cd.compile_dfa(aut.V, aut.S, aut.start, aut.row_ptr, aut.tok, aut.next, aut.accepting, device="cuda:0")
    x = [torch.zeros((4, 64), device="cuda:0")]
    counter = torch.zeros(1, dtype=torch.int32, device="cuda:0")
    with pytest.raises(cd.CdError) as e:  # cd_set_satisfying not called
        cd.decode_loop(dfa, x, limit=1, satisfied=counter)
    assert e.value.code == 1
    dfa.set_satisfying([0, 1])
    with pytest.raises(cd.CdError) as e:
        cd.decode_loop(dfa, x, limit=-1, satisfied=counter)
    assert e.value.code == 1
    out = cd.decode_loop(dfa, x, limit=2, satisfied=counter)
    assert int(counter) == 4 and bool(out["done"].all())  # rows finishing in the same step are all kept
    dfa.close()


def test_host_buffer_loop_matches_device_loop(cd, oracle):
    cfg = wl.scaled(wl.CONFIGS["c3"], V=30000, B=300, S=64, max_steps=8)
    aut = wl.build_automaton(cfg, device="cuda:0")
    logits = wl.build_step_logits(cfg, aut, device="cuda:0")
    dfa = dev_dfa(cd, aut)
    out = cd.decode_loop(dfa, logits, max_steps=cfg.max_steps)
    # pinned, device-mapped buffers (the SMs pull the active rows over PCIe) and pageable buffers
    # (cudaMemcpyAsync per run of active rows) take different paths inside the library
    for host in ([x.cpu().pin_memory() for x in logits], [x.cpu() for x in logits]):
        out_h = cd.decode_loop_host(dfa, host, max_steps=cfg.max_steps)
        for k in ("tokens", "len", "final_state", "done", "sum_logprob"):
            assert torch.equal(out[k].cpu(), out_h[k]), k
    dfa.close()


def test_host_buffer_loop_gathers_over_the_link_in_automatic_mode(cd, oracle):
    """cd_decode_loop_host with cd_set_gather_max(-1) and pinned, mapped buffers: every state of this automaton has fewer
    than V / 32 transitions, so the step kernel reads the allowed logits straight from host memory (nothing is staged);
    with pageable buffers the same call stages the active rows.  Both against the oracle."""
    cfg = wl.scaled(wl.CONFIGS["c3"], V=30000, B=300, S=64, max_steps=8)
    aut = wl.build_automaton(cfg)
    assert int(torch.diff(torch.as_tensor(aut.row_ptr)).max()) <= cfg.V // 32
    logits = wl.build_step_logits(cfg, aut, device="cuda:0")
    want = oracle.decode_loop(aut, [x.cpu() for x in logits])
    dfa = cd.compile_dfa(aut.V, aut.S, aut.start, aut.row_ptr, aut.tok, aut.next, aut.accepting, device="cuda:0")
    dfa.set_gather_max(-1)
    for host in ([x.cpu().pin_memory() for x in logits], [x.cpu() for x in logits]):
        got = cd.decode_loop_host(dfa, host, max_steps=cfg.max_steps)
        for k in ("tokens", "len", "final_state", "done"):
            assert np.array_equal(got[k].numpy(), want[k]), k
        ok, worst = close(got["sum_logprob"].numpy(), want["sum_logprob"], tol=TOL * cfg.max_steps)
        assert ok, worst
    dfa.close()


def test_trie_sugar_equals_explicit_csr(cd, oracle):
    cfg = wl.scaled(wl.CONFIGS["c2"], V=20000, B=200, K=30)
    aut = wl.build_automaton(cfg)
    logits = wl.build_step_logits(cfg, aut, device="cuda:0")
    d1 = dev_dfa(cd, aut)
    d2 = cd.compile_trie(cfg.V, aut.labels, device="cuda:0")
    apply_mode(d2, aut)
    assert (d1.S, d1.nnz) == (d2.S, d2.nnz)
    o1 = cd.decode_loop(d1, logits)
    o2 = cd.decode_loop(d2, logits)
    for k in o1:
        assert torch.equal(o1[k], o2[k])
    d1.close()
    d2.close()


def test_stepwise_api_reproduces_the_loop(cd, oracle):
    cfg = wl.scaled(wl.CONFIGS["c3"], V=70000, B=700, S=128, max_steps=12)
    aut = wl.build_automaton(cfg, device="cuda:0")
    logits = wl.build_step_logits(cfg, aut, device="cuda:0")
    dfa = dev_dfa(cd, aut)
    out = cd.decode_loop(dfa, logits)
    ids = torch.arange(cfg.B, dtype=torch.int32, device="cuda:0")
    st = torch.full((cfg.B,), aut.start, dtype=torch.int32, device="cuda:0")
    toks = torch.full((cfg.B, cfg.max_steps), -1, dtype=torch.int32, device="cuda:0")
    n = cfg.B
    for k in range(cfg.max_steps):
        if n == 0:
            break
        tok, lp, lse, done = cd.step(dfa, logits[k], st, row_map=ids, n=n)
        toks[ids[:n].long(), k] = tok
        ids, st, na = cd.compact(done, ids, st, n=n)
        n = int(na)
    assert torch.equal(toks, out["tokens"])
    dfa.close()


def test_two_streams_share_one_handle(cd, oracle):
    """include/cd.h: a handle may be used from several streams at once (scratch is kept per
    (handle, stream)).  Two loops on two streams, interleaved launches, different inputs."""
    cfg = wl.scaled(wl.CONFIGS["c3"], V=20000, B=200, S=40, max_steps=6)
    aut = wl.build_automaton(cfg)
    dfa = dev_dfa(cd, aut)
    la = wl.build_step_logits(cfg, aut, device="cuda:0", batch=0)
    lb = wl.build_step_logits(cfg, aut, device="cuda:0", batch=1)
    torch.cuda.synchronize()
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    outs = {}
    for rep in range(3):
        with torch.cuda.stream(s1):
            outs["a"] = cd.decode_loop(dfa, la)
        with torch.cuda.stream(s2):
            outs["b"] = cd.decode_loop(dfa, lb)
    torch.cuda.synchronize()
    for key, logits in (("a", la), ("b", lb)):
        want = oracle.decode_loop(aut, [x.cpu() for x in logits])
        for k in ("tokens", "len", "final_state", "done"):
            assert np.array_equal(outs[key][k].cpu().numpy(), want[k]), (key, k)


def test_step_and_compact_in_a_cuda_graph(cd, oracle):
    """cd_step / cd_compact neither allocate nor synchronise after cd_reserve, so a decoding step
    can be captured in a CUDA graph and replayed on new inputs written into the same buffers."""
    cfg = wl.scaled(wl.CONFIGS["c3"], V=20000, B=96, S=40, max_steps=1)
    aut = wl.build_automaton(cfg)
    dfa = dev_dfa(cd, aut)
    n = cfg.B
    x = torch.empty((n, cfg.V), dtype=torch.bfloat16, device="cuda:0")
    st = torch.empty(n, dtype=torch.int32, device="cuda:0")
    outb = (torch.empty(n, dtype=torch.int32, device="cuda:0"), torch.empty(n, dtype=torch.float32, device="cuda:0"),
            torch.empty(n, dtype=torch.float32, device="cuda:0"), torch.empty(n, dtype=torch.uint8, device="cuda:0"))
    cmp_out = (torch.empty(n, dtype=torch.int32, device="cuda:0"), torch.empty(n, dtype=torch.int32, device="cuda:0"),
               torch.empty(1, dtype=torch.int32, device="cuda:0"))
    acc = np.asarray(aut.accepting)
    live = [s for s in range(aut.S) if not acc[s]]
    side = torch.cuda.Stream()
    with torch.cuda.stream(side):
        dfa.reserve(n)
        st.fill_(live[0])
        x.zero_()
        cd.step(dfa, x, st, out=outb)  # warm-up on the capture stream: scratch + kernel attributes
        cd.compact(outb[3], None, st, out=cmp_out)
        side.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=side):
            cd.step(dfa, x, st, out=outb)
            cd.compact(outb[3], None, st, out=cmp_out)
    torch.cuda.synchronize()
    for rep in range(3):
        logits = wl.make_logits(100 + rep, 0, n, cfg.V, 3.0, torch.bfloat16)
        states = [live[(i + rep) % len(live)] for i in range(n)]
        x.copy_(logits)
        st.copy_(torch.tensor(states, dtype=torch.int32))
        torch.cuda.synchronize()
        g.replay()
        torch.cuda.synchronize()
        o_tok, o_lp, o_lse, o_done, o_st = oracle.step(aut, logits, states)
        assert outb[0].cpu().numpy().tolist() == o_tok.tolist()
        assert st.cpu().numpy().tolist() == o_st.tolist()
        o_ro, o_so, k = oracle.compact(o_done, None, o_st)
        assert int(cmp_out[2]) == k and cmp_out[0][:k].cpu().numpy().tolist() == o_ro.tolist()


def test_loop_many_rows_small_vocab(cd, oracle):
    """B = 10,000 rows (more than one chunk of the one-CTA compaction, more rows than the c4 batch)
    at a small vocabulary: the fused loop end to end against the oracle."""
    cfg = wl.scaled(wl.CONFIGS["c3"], V=2048, B=10000, S=24, max_steps=6, density=0.05)
    aut = wl.build_automaton(cfg)
    dfa = dev_dfa(cd, aut)
    logits = wl.build_step_logits(cfg, aut, device="cuda:0")
    got = cd.decode_loop(dfa, logits)
    torch.cuda.synchronize()
    want = oracle.decode_loop(aut, [x.cpu() for x in logits])
    for k in ("tokens", "len", "final_state", "done"):
        assert np.array_equal(got[k].cpu().numpy(), want[k]), k
    ok, worst = close(got["sum_logprob"].cpu().numpy(), want["sum_logprob"], tol=TOL * cfg.max_steps)
    assert ok, worst
    assert want["n_active_hist"][1] > 4096  # the second step still compacts more than one chunk
