"""Pins for the CPU oracle (oracle/oracle_cd.c) against things other than itself.

The paper prints no worked numeric example of a decoding step (SURVEY.md
section 4), so the pins are: library routines on the special case that reduces
to a textbook op, closed forms, brute force written a different way, the
language of the automaton, and invariants (SURVEY.md 8(c) "What pins each
part").  Each is chosen so that one plausible mistake (dropped mask, wrong tie
rule, sum over the wrong set, m - lse cancellation, wrong CSR pairing,
unstable compaction, advancing an accepted row) fails it.
"""
import math

import numpy as np
import pytest
import torch

import workloads as wl


class Aut:
    """Minimal host CSR holder (so tests can hand-build automata)."""

    def __init__(self, V, rows, accepting, start=0):
        # rows: list (per state) of sorted [(tok, next), ...]
        self.V, self.S, self.start = V, len(rows), start
        rp, tk, nx = [0], [], []
        for r in rows:
            for t, n in r:
                tk.append(t)
                nx.append(n)
            rp.append(len(tk))
        self.row_ptr = np.array(rp, np.int64)
        self.tok = np.array(tk, np.int32)
        self.next = np.array(nx, np.int32)
        self.accepting = np.array(accepting, np.uint8)


def all_ones(V):
    """state 0 allows every token -> state 1 (accepting leaf)."""
    return Aut(V, [[(t, 1) for t in range(V)], []], [0, 1])


def subset(V, toks, nxt=1):
    return Aut(V, [[(t, nxt) for t in sorted(toks)], []], [0, 1])


# ---------------------------------------------------------------- library pin
@pytest.mark.parametrize("V", [32, 1000, 4096])
def test_all_ones_mask_is_textbook_log_softmax_fp32(oracle, V):
    g = torch.Generator().manual_seed(100 + V)
    x = torch.randn(7, V, generator=g) * 3.0
    # library argmax tie rules may differ from ours: keep the maximum unique here
    assert all(int((r == r.max()).sum()) == 1 for r in x)
    tok, lp, lse, done, st = oracle.step(all_ones(V), x, [0] * 7)
    ref_ls = torch.log_softmax(x.double(), dim=1)
    ref_arg = torch.argmax(x, dim=1)
    assert tok.tolist() == ref_arg.tolist()
    np.testing.assert_allclose(lp, ref_ls[torch.arange(7), ref_arg].numpy(), rtol=0, atol=1e-12)
    np.testing.assert_allclose(lse, torch.logsumexp(x.double(), dim=1).numpy(), rtol=1e-13, atol=1e-12)
    assert done.tolist() == [1] * 7 and st.tolist() == [1] * 7


def test_all_ones_mask_bf16_widening_is_exact(oracle):
    V = 2048
    g = torch.Generator().manual_seed(5)
    x = (torch.randn(5, V, generator=g) * 2.0).to(torch.bfloat16)
    x[:, 77] = 30.0  # unique maximum so library argmax tie rules do not matter
    tok, lp, lse, _, _ = oracle.step(all_ones(V), x, [0] * 5)
    xd = x.float().double()  # bf16 -> fp32 is exact
    assert tok.tolist() == [77] * 5
    np.testing.assert_allclose(lse, torch.logsumexp(xd, dim=1).numpy(), rtol=1e-13)
    np.testing.assert_allclose(lp, torch.log_softmax(xd, dim=1)[:, 77].numpy(), atol=1e-12)


# ---------------------------------------------------------------- closed forms
def test_single_allowed_token_is_forced(oracle):
    V = 512
    x = torch.randn(3, V, generator=torch.Generator().manual_seed(1))
    x[:, 400] = -7.25  # far from the row maximum
    tok, lp, lse, done, st = oracle.step(subset(V, [400]), x, [0, 0, 0])
    assert tok.tolist() == [400] * 3
    assert lp.tolist() == [0.0] * 3  # exactly zero
    assert lse.tolist() == [-7.25] * 3


@pytest.mark.parametrize("a,b", [(0.5, -1.25), (-3.0, -3.0), (10.0, 9.0), (-20.0, 1.0), (0.0, 20.0)])
def test_two_allowed_tokens_closed_form(oracle, a, b):
    V = 64
    x = torch.full((1, V), 50.0)  # disallowed logits are huge: dropping the mask fails
    x[0, 9], x[0, 41] = a, b
    tok, lp, lse, _, _ = oracle.step(subset(V, [9, 41]), x, [0])
    assert tok[0] == (9 if a >= b else 41)  # tie -> lowest id
    assert lp[0] == pytest.approx(-math.log1p(math.exp(-abs(a - b))), abs=1e-14)
    assert lse[0] == pytest.approx(max(a, b) + math.log1p(math.exp(-abs(a - b))), abs=1e-13)


def test_cancellation_free_logprob_near_zero(oracle):
    # two tokens 20 apart: log p = -log1p(e^-20) ~ -2.06e-9; (m - lse) in fp32 would give 0
    V = 64
    x = torch.zeros((1, V))
    x[0, 3], x[0, 5] = 100.0, 80.0
    _, lp, _, _, _ = oracle.step(subset(V, [3, 5]), x, [0])
    assert lp[0] == pytest.approx(-math.log1p(math.exp(-20.0)), rel=1e-12)
    assert lp[0] < 0.0


@pytest.mark.parametrize("k", [2, 3, 5, 50])
def test_k_equal_logits(oracle, k):
    V = 1024
    ids = sorted(np.random.default_rng(k).choice(V, size=k, replace=False).tolist())
    x = torch.randn(1, V, generator=torch.Generator().manual_seed(k)) + 9.0
    x[0, ids] = 1.5
    tok, lp, lse, _, _ = oracle.step(subset(V, ids), x, [0])
    assert tok[0] == ids[0]
    assert lp[0] == pytest.approx(-math.log(k), abs=1e-14)
    assert lse[0] == pytest.approx(1.5 + math.log(k), abs=1e-13)


# ---------------------------------------------------------------- brute force
def _brute_step(aut, x_row, s):
    """Same quantity, written a third way: python sets, fsum, explicit tie set."""
    lo, hi = int(aut.row_ptr[s]), int(aut.row_ptr[s + 1])
    trans = {int(aut.tok[j]): int(aut.next[j]) for j in range(lo, hi)}
    allowed = set(trans)
    vals = {t: float(x_row[t]) for t in range(aut.V) if t in allowed}
    m = max(vals.values())
    tstar = min(t for t, v in vals.items() if v == m)
    z = math.fsum(math.exp(v - m) for v in vals.values())
    return tstar, -math.log(z), m + math.log(z), trans[tstar]


@pytest.mark.parametrize("dtype", [torch.float32, torch.bfloat16])
@pytest.mark.parametrize("V,S,density", [(64, 5, 0.3), (256, 9, 0.05), (1024, 16, 0.02)])
def test_brute_force_tiny_vocab(oracle, dtype, V, S, density):
    aut = wl.make_random_dfa(seed=V + S, V=V, S=S, density=density, accept_frac=0.3)
    assert oracle.validate(aut) == 0
    n = 40
    g = torch.Generator().manual_seed(V)
    x = (torch.randn(n, V, generator=g) * 2.0).to(dtype)  # bf16 at std 2 has natural ties
    live = [s for s in range(S) if not aut.accepting[s]]
    states = [live[i % len(live)] for i in range(n)]
    tok, lp, lse, done, st = oracle.step(aut, x, states)
    xf = x.float().numpy()
    for i in range(n):
        t, l, z, ns = _brute_step(aut, xf[i], states[i])
        assert tok[i] == t
        assert st[i] == ns
        assert done[i] == int(aut.accepting[ns])
        assert lp[i] == pytest.approx(l, abs=1e-12)
        assert lse[i] == pytest.approx(z, abs=1e-12)


# ---------------------------------------------------------------- mask really masks
def test_poisoned_complement_changes_nothing(oracle):
    V = 1024
    aut = wl.make_random_dfa(seed=7, V=V, S=6, density=0.04, accept_frac=0.2)
    g = torch.Generator().manual_seed(3)
    x = torch.randn(12, V, generator=g)
    live = [s for s in range(aut.S) if not aut.accepting[s]]
    states = [live[i % len(live)] for i in range(12)]
    base = oracle.step(aut, x, states)
    for poison in (1e30, float("inf"), float("nan"), -float("inf")):
        y = x.clone()
        for i, s in enumerate(states):
            lo, hi = int(aut.row_ptr[s]), int(aut.row_ptr[s + 1])
            dis = torch.ones(V, dtype=torch.bool)
            dis[aut.tok[lo:hi].long()] = False
            y[i, dis] = poison
        out = oracle.step(aut, y, states)
        for a, b in zip(base, out):
            assert np.array_equal(a, b)


def test_adversarial_mass_on_disallowed_still_yields_a_label(oracle):
    # with options, the result is always a value in the option set
    cfg = wl.scaled(wl.CONFIGS["c2"], V=4096, B=64, K=12)
    aut = wl.build_automaton(cfg)
    logits = wl.build_step_logits(cfg, aut)
    allowed_anywhere = set(aut.tok.tolist())
    for x in logits:
        bad = torch.ones(cfg.V, dtype=torch.bool)
        bad[list(allowed_anywhere)] = False
        x[:, bad] += 40.0
    res = oracle.decode_loop(aut, logits)
    labels = {tuple(l) for l in aut.labels}
    for r in range(cfg.B):
        assert res["done"][r] == 1
        assert tuple(res["tokens"][r, : res["len"][r]].tolist()) in labels


# ---------------------------------------------------------------- tie rule
def test_planted_ties_pick_lowest_id(oracle):
    V = 4096
    for ids in ([31, 32], [255, 256, 257], [0, V - 1], [1023, 1024, 2047, 2048, 4095]):
        x = torch.randn(1, V, generator=torch.Generator().manual_seed(len(ids))).clamp_(max=3.0)
        x[0, ids] = 3.5
        tok, lp, _, _, _ = oracle.step(all_ones(V), x, [0])
        assert tok[0] == ids[0]
        # and when the lowest planted id is not allowed, the next one wins
        tok2, _, _, _, _ = oracle.step(subset(V, [t for t in range(V) if t != ids[0]]), x, [0])
        assert tok2[0] == ids[1]


def test_signed_zero_ties(oracle):
    V = 64
    x = torch.full((1, V), -1.0)
    x[0, 5], x[0, 9] = -0.0, 0.0  # equal under float comparison -> lowest id
    tok, _, _, _, _ = oracle.step(all_ones(V), x, [0])
    assert tok[0] == 5


# ---------------------------------------------------------------- invariants
@pytest.mark.parametrize("dtype", [torch.float32, torch.bfloat16])
def test_invariants_on_random_dfa(oracle, dtype):
    V, S, n = 2048, 32, 64
    aut = wl.make_random_dfa(seed=11, V=V, S=S, density=0.03, accept_frac=0.1)
    x = (torch.randn(n, V, generator=torch.Generator().manual_seed(2)) * 3.0).to(dtype)
    live = [s for s in range(S) if not aut.accepting[s]]
    states = [live[(7 * i) % len(live)] for i in range(n)]
    tok, lp, lse, done, st = oracle.step(aut, x, states)
    xd = x.float().double()
    full = torch.logsumexp(xd, dim=1).numpy()
    for i, s in enumerate(states):
        lo, hi = int(aut.row_ptr[s]), int(aut.row_ptr[s + 1])
        A = aut.tok[lo:hi].long()
        assert tok[i] in set(A.tolist())  # chosen token always allowed
        assert lp[i] <= 0.0
        assert lse[i] <= full[i] + 1e-12  # masking removes mass
        p = torch.exp(xd[i, A] - lse[i])
        assert abs(float(p.sum()) - 1.0) < 1e-6  # exp(logprobs) over allowed sums to 1
        assert float(xd[i, tok[i]]) - lse[i] == pytest.approx(lp[i], abs=1e-9)
    # shift invariance: token, state, done identical; logprob unchanged; lse shifts
    x2 = (x.float() + 8.0).to(dtype) if dtype == torch.float32 else (x.float() * 1.0).to(dtype)
    if dtype == torch.float32:
        tok2, lp2, lse2, done2, st2 = oracle.step(aut, x2, states)
        assert tok2.tolist() == tok.tolist() and st2.tolist() == st.tolist()
        np.testing.assert_allclose(lp2, lp, atol=2e-5)
        np.testing.assert_allclose(lse2, lse + 8.0, atol=2e-5)


def test_row_independence_and_row_map(oracle):
    V, S, n = 1024, 12, 33
    aut = wl.make_random_dfa(seed=21, V=V, S=S, density=0.05, accept_frac=0.2)
    x = torch.randn(n, V, generator=torch.Generator().manual_seed(9)).to(torch.bfloat16)
    live = [s for s in range(S) if not aut.accepting[s]]
    states = np.array([live[i % len(live)] for i in range(n)], np.int32)
    base = oracle.step(aut, x, states)
    perm = np.random.default_rng(0).permutation(n)
    out = oracle.step(aut, x, states[perm], row_map=perm)  # slot i reads row perm[i]
    for a, b in zip(base, out):
        assert np.array_equal(a[perm], b)
    out2 = oracle.step(aut, x[torch.from_numpy(perm)], states[perm])  # physically shuffled
    for a, b in zip(out, out2):
        assert np.array_equal(a, b)


def test_row_stride_ld_greater_than_V(oracle):
    V, ld = 96, 128
    aut = wl.make_random_dfa(seed=2, V=V, S=4, density=0.2, accept_frac=0.25)
    x = torch.randn(6, ld, generator=torch.Generator().manual_seed(4))
    x[:, V:] = 99.0  # padding must never be read
    live = [s for s in range(aut.S) if not aut.accepting[s]]
    states = [live[i % len(live)] for i in range(6)]
    a = oracle.step(aut, x, states)
    b = oracle.step(aut, x[:, :V].contiguous(), states)
    for u, v in zip(a, b):
        assert np.array_equal(u, v)


def test_nan_and_minus_inf(oracle):
    V = 64
    ids = [4, 8, 15, 16]
    x = torch.zeros((3, V))
    x[0, ids] = torch.tensor([float("nan"), 1.0, float("nan"), 1.0])  # NaN == -inf
    x[1, ids] = torch.tensor([-float("inf")] * 4)  # all -inf: lowest allowed id, -inf
    x[2, ids] = torch.tensor([-float("inf"), 2.0, 2.0, -float("inf")])
    tok, lp, lse, done, st = oracle.step(subset(V, ids), x, [0, 0, 0])
    assert tok.tolist() == [8, 4, 8]
    assert lp[0] == pytest.approx(-math.log(2.0), abs=1e-15)
    assert lp[1] == -math.inf and lse[1] == -math.inf
    assert lp[2] == pytest.approx(-math.log(2.0), abs=1e-15)
    assert done.tolist() == [1, 1, 1]


def test_plus_inf_token_is_lowest_inf_id(oracle):
    V = 64
    x = torch.zeros((1, V))
    x[0, 20] = x[0, 10] = float("inf")
    tok, _, _, _, _ = oracle.step(all_ones(V), x, [0])
    assert tok[0] == 10  # value outputs are unspecified here (G6): parity unpinned


# ---------------------------------------------------------------- accepted rows
def test_accepted_rows_never_advance(oracle):
    V = 64
    aut = Aut(V, [[(3, 1)], [(5, 0)]], [0, 1])  # state 1 accepts but HAS a transition
    x = torch.randn(2, V, generator=torch.Generator().manual_seed(0))
    tok, lp, lse, done, st = oracle.step(aut, x, [1, 0])
    assert tok.tolist() == [-1, 3]
    assert st.tolist() == [1, 1]
    assert done.tolist() == [1, 1]
    assert lp[0] == 0.0


# ---------------------------------------------------------------- validation
def test_validate_codes(oracle):
    ok = Aut(16, [[(1, 1), (4, 0)], []], [0, 1])
    assert oracle.validate(ok) == 0
    bad = Aut(16, [[(4, 1), (1, 0)], []], [0, 1])  # not strictly increasing
    assert oracle.validate(bad) == 2
    dup = Aut(16, [[(4, 1), (4, 0)], []], [0, 1])
    assert oracle.validate(dup) == 2
    oob = Aut(16, [[(16, 1)], []], [0, 1])
    assert oracle.validate(oob) == 2
    oobn = Aut(16, [[(3, 2)], []], [0, 1])
    assert oracle.validate(oobn) == 2
    dead = Aut(16, [[(3, 1)], []], [0, 0])  # non-accepting state without transitions
    assert oracle.validate(dead) == 3
    leaf = Aut(16, [[(3, 1)], []], [0, 1])  # accepting leaf is fine
    assert oracle.validate(leaf) == 0
    st = Aut(16, [[(3, 1)], []], [0, 1], start=2)
    assert oracle.validate(st) == 2
    rp = Aut(16, [[(3, 1)], []], [0, 1])
    rp.row_ptr = np.array([0, 2, 1], np.int64)
    assert oracle.validate(rp) == 2


# ---------------------------------------------------------------- compaction
@pytest.mark.parametrize("n", [0, 1, 2, 31, 32, 33, 1000, 1024, 1025, 4097])
@pytest.mark.parametrize("pattern", ["none", "all", "alt", "rand"])
def test_compaction_is_stable_filter(oracle, n, pattern):
    rng = np.random.default_rng(n)
    done = {
        "none": np.zeros(n, np.uint8),
        "all": np.ones(n, np.uint8),
        "alt": (np.arange(n) % 2).astype(np.uint8),
        "rand": (rng.random(n) < 0.3).astype(np.uint8),
    }[pattern]
    ids = np.sort(rng.choice(10 * n + 1, size=n, replace=False)).astype(np.int32)
    st = rng.integers(0, 1000, size=n).astype(np.int32)
    ro, so, k = oracle.compact(done, ids, st)
    keep = [i for i in range(n) if not done[i]]
    assert k == len(keep) == n - int(done.sum())
    assert ro.tolist() == [int(ids[i]) for i in keep]
    assert so.tolist() == [int(st[i]) for i in keep]
    assert all(ro[i] < ro[i + 1] for i in range(k - 1))  # ascending stays ascending
    ro2, _, k2 = oracle.compact(done)  # implicit ids 0..n-1
    assert ro2.tolist() == keep and k2 == k


# ---------------------------------------------------------------- the loop
def test_config_c0_by_hand(oracle):
    """BASELINE.json configs[0]: language {[17,3],[42]}.  Every row is computable
    from three logits (SURVEY 8(c) pin table)."""
    cfg = wl.CONFIGS["c0"]
    aut = wl.build_automaton(cfg)
    assert aut.S == 4 and aut.tok.tolist() == [17, 42, 3] and aut.accepting.tolist() == [0, 0, 1, 1]
    logits = wl.build_step_logits(cfg, aut)
    res = oracle.decode_loop(aut, logits)
    for r in range(cfg.B):
        a, b = float(logits[0][r, 17]), float(logits[0][r, 42])
        lp0 = -math.log1p(math.exp(-abs(a - b)))
        if a >= b:
            assert res["tokens"][r].tolist() == [17, 3] + [-1] * 6
            assert res["len"][r] == 2 and res["final_state"][r] == 2
        else:
            assert res["tokens"][r].tolist() == [42] + [-1] * 7
            assert res["len"][r] == 1 and res["final_state"][r] == 3
        assert res["done"][r] == 1
        assert res["sum_logprob"][r] == pytest.approx(lp0, abs=1e-14)  # step 1 is forced: +0
    hist = res["n_active_hist"].tolist()
    n17 = sum(1 for r in range(cfg.B) if float(logits[0][r, 17]) >= float(logits[0][r, 42]))
    assert hist == [cfg.B, n17] + [0] * 6


def _enumerate_language(aut, limit=10000):
    """Every string the automaton accepts under shortest-accept semantics."""
    out, stack = [], [(aut.start, [])]
    while stack:
        s, pre = stack.pop()
        if aut.accepting[s]:
            out.append(tuple(pre))
            continue
        for j in range(int(aut.row_ptr[s]), int(aut.row_ptr[s + 1])):
            stack.append((int(aut.next[j]), pre + [int(aut.tok[j])]))
        assert len(out) < limit
    return out


@pytest.mark.parametrize("name,V,B,K", [("c1", 8192, 64, 2), ("c2", 8192, 96, 50)])
def test_trie_decodes_only_labels(oracle, name, V, B, K):
    cfg = wl.scaled(wl.CONFIGS[name], V=V, B=B, K=K)
    aut = wl.build_automaton(cfg)
    assert oracle.validate(aut) == 0
    lang = _enumerate_language(aut)
    assert sorted(lang) == sorted(tuple(l) for l in aut.labels)  # the K labels, nothing else
    logits = wl.build_step_logits(cfg, aut)
    res = oracle.decode_loop(aut, logits)
    leaf = {tuple(l): aut.leaf_of_label[i] for i, l in enumerate(aut.labels)}
    assert res["done"].all()  # max_steps = longest label
    for r in range(B):
        h = tuple(res["tokens"][r, : res["len"][r]].tolist())
        assert h in leaf and res["final_state"][r] == leaf[h]
        assert (res["tokens"][r, res["len"][r]:] == -1).all()
    # greedy per step: the first token is the best allowed first token (two-level check)
    first = sorted({l[0] for l in aut.labels})
    x0 = logits[0].float()
    for r in range(B):
        vals = x0[r, first]
        best = first[int(torch.nonzero(vals == vals.max())[0])]
        assert res["tokens"][r, 0] == best


def test_random_dfa_replay_and_freeze(oracle):
    cfg = wl.scaled(wl.CONFIGS["c3"], V=4096, B=128, S=64, max_steps=12)
    aut = wl.build_automaton(cfg)
    logits = wl.build_step_logits(cfg, aut)
    res = oracle.decode_loop(aut, logits)
    trans = {}
    for s in range(aut.S):
        for j in range(int(aut.row_ptr[s]), int(aut.row_ptr[s + 1])):
            trans[(s, int(aut.tok[j]))] = int(aut.next[j])
    n_hist = [0] * cfg.max_steps
    for r in range(cfg.B):
        s, k = aut.start, 0
        while k < cfg.max_steps and not aut.accepting[s]:
            n_hist[k] += 1
            t = int(res["tokens"][r, k])
            assert (s, t) in trans  # token allowed in the state the row was in
            s = trans[(s, t)]
            k += 1
        assert res["len"][r] == k and res["final_state"][r] == s
        assert res["done"][r] == int(aut.accepting[s])
        assert (res["tokens"][r, k:] == -1).all()  # frozen after accept
    assert res["n_active_hist"].tolist() == n_hist
    # stepwise API reproduces the loop (step + compact composed by hand)
    ids = np.arange(cfg.B, dtype=np.int32)
    st = np.full(cfg.B, aut.start, np.int32)
    slp = np.zeros(cfg.B)
    for k in range(cfg.max_steps):
        if len(ids) == 0:
            break
        tok, lp, lse, done, st = oracle.step(aut, logits[k], st, row_map=ids)
        assert tok.tolist() == res["tokens"][ids, k].tolist()
        slp[ids] += lp
        ids, st, _ = oracle.compact(done, ids, st)
    np.testing.assert_allclose(slp, res["sum_logprob"], atol=1e-12)


def test_accepting_start_returns_all_done(oracle):
    aut = Aut(32, [[(1, 0)]], [1])
    x = [torch.zeros(3, 32)]
    res = oracle.decode_loop(aut, x)
    assert res["done"].tolist() == [1, 1, 1] and res["len"].tolist() == [0, 0, 0]
    assert (res["tokens"] == -1).all()


def test_survival_statistics_sanity(oracle):
    # SURVEY 8(c) "statistics": active fraction after k steps ~ (1 - accept_frac)^k
    cfg = wl.scaled(wl.CONFIGS["c3"], V=2048, B=2000, S=256, max_steps=6, density=0.05)
    aut = wl.build_automaton(cfg)
    logits = wl.build_step_logits(cfg, aut)
    res = oracle.decode_loop(aut, logits)
    acc = float(aut.accepting.float().mean())
    for k, n in enumerate(res["n_active_hist"].tolist()):
        expect = cfg.B * (1 - acc) ** k
        assert abs(n - expect) < 6 * math.sqrt(cfg.B) + 0.1 * expect
