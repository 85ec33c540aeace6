"""Pins for the oracle's LM-head step (oracle_cd.c O6) against things
other than itself:

  * exact-arithmetic inputs (multiples of 1/8): the logits are exactly representable in
    fp32, so O6 must equal the already pinned O2 (oracle.step) applied to logits formed
    by a LIBRARY matmul (numpy float64) -- token, state, done identical, logprob / lse to
    1e-12;
  * the all-ones automaton reduces to the textbook log_softmax / argmax of hidden @ W.T
    (torch float64);
  * closed forms: one-hot embedding rows (logit = one hidden component), a single allowed
    token, two allowed tokens (-log1p(exp(-|d|))), k identical embedding rows (-log k,
    lowest id);
  * a non-square W with padded strides catches a transposed operand or a wrong stride;
  * rows are independent and row_map only selects the hidden row.
"""
import math

import numpy as np
import pytest
import torch

import workloads as wl


def all_ones_automaton(V):
    """One non-accepting state allowing every token, all leading to an accepting sink."""
    rp = torch.tensor([0, V, V], dtype=torch.int64)
    tok = torch.arange(V, dtype=torch.int32)
    nxt = torch.ones(V, dtype=torch.int32)
    acc = torch.tensor([0, 1], dtype=torch.uint8)
    return wl.Automaton(V=V, S=2, start=0, row_ptr=rp, tok=tok, next=nxt, accepting=acc)


def f64(x):
    return x.to(torch.float64).numpy()


@pytest.mark.parametrize("seed,V,H,S", [(1, 300, 64, 7), (2, 1024, 200, 16), (3, 257, 33, 5)])
def test_exact_inputs_reduce_to_step_on_library_matmul(oracle, seed, V, H, S):
    aut = wl.make_random_dfa(seed, V, S, 0.3, 0.2)
    B = 19
    hid = wl.make_hidden(seed, 0, B, H, exact=True, ld=H + 8)
    W = wl.make_head(seed, V, H, 2.0, exact=True, ld=H + 16)
    x = f64(hid[:, :H]) @ f64(W[:, :H]).T  # library matmul, float64
    x32 = x.astype(np.float32)
    assert np.array_equal(x32.astype(np.float64), x)  # exactly representable
    state = [(r * 3) % S for r in range(B)]
    state = [s if not int(aut.accepting[s]) else 0 for s in state]
    tk, lp, lse, dn, st, gap = oracle.head_step(aut, hid, W, H, state)
    tk2, lp2, lse2, dn2, st2 = oracle.step(aut, x32, state)
    assert np.array_equal(tk, tk2) and np.array_equal(st, st2) and np.array_equal(dn, dn2)
    assert np.allclose(lp, lp2, rtol=0, atol=1e-12) and np.allclose(lse, lse2, rtol=1e-13, atol=1e-12)
    assert (gap >= 0).all()


def test_all_ones_is_textbook_log_softmax(oracle):
    V, H, B = 500, 48, 8
    aut = all_ones_automaton(V)
    hid = wl.make_hidden(5, 0, B, H)
    W = wl.make_head(5, V, H, 2.0)
    x = torch.from_numpy(f64(hid) @ f64(W).T)
    ls = torch.log_softmax(x, dim=1)
    want_tok = torch.argmax(x, dim=1).numpy()
    tk, lp, lse, dn, st, gap = oracle.head_step(aut, hid, W, H, [0] * B)
    assert np.array_equal(tk, want_tok)  # gaussian data: tie-free
    assert np.allclose(lp, ls.max(dim=1).values.numpy(), rtol=0, atol=1e-12)
    assert np.allclose(lse, torch.logsumexp(x, dim=1).numpy(), rtol=1e-13, atol=1e-12)
    assert (dn == 1).all() and (st == 1).all()
    # gap = best - second best
    top2 = torch.topk(x, 2, dim=1).values
    assert np.allclose(gap, (top2[:, 0] - top2[:, 1]).numpy(), rtol=0, atol=1e-12)


def test_one_hot_rows_pick_hidden_components(oracle):
    # W[t] = e_{t mod H}: logit of token t is hidden[t mod H]; non-square, padded strides
    V, H, B = 40, 12, 3
    W = torch.zeros((V, H + 4), dtype=torch.bfloat16)
    for t in range(V):
        W[t, t % H] = 1.0
    W[:, H:] = 7.0  # padding must not be read
    hid = torch.zeros((B, H + 2), dtype=torch.bfloat16)
    hid[:, :H] = torch.tensor([[0.5, -1, 2, 3, -4, 0.25, 1, 1.5, -0.5, 0, 2.5, -2]] * B, dtype=torch.bfloat16)
    hid[1, 3] = -8.0  # row 1: component 3 is no longer the best
    hid[:, H:] = 9.0
    aut = all_ones_automaton(V)
    tk, lp, lse, dn, st, gap = oracle.head_step(aut, hid, W, H, [0] * B)
    # row 0/2: best component is 3 (value 3.0): tokens 3, 15, 27, 39 tie -> lowest id 3
    assert tk[0] == 3 and tk[2] == 3 and gap[0] == 0.0
    assert tk[1] == 10  # 2.5 at component 10
    vals = f64(hid[0, :H])
    per_tok = np.array([vals[t % H] for t in range(V)])
    want = math.log(np.exp(per_tok - 3.0).sum())
    assert abs(lp[0] + want) < 1e-12 and abs(lse[0] - (3.0 + want)) < 1e-12
    assert oracle.head_logit(hid, W, H, 1, 15) == -8.0


def test_closed_forms_and_row_map(oracle):
    V, H = 64, 16
    hid = wl.make_hidden(9, 0, 6, H)
    W = wl.make_head(9, V, H, 3.0)
    # state 0: single token 5; state 1: tokens {7, 20}; state 2: tokens {30, 31, 32}; state 3 accepting
    rp = torch.tensor([0, 1, 3, 6, 6], dtype=torch.int64)
    tok = torch.tensor([5, 7, 20, 30, 31, 32], dtype=torch.int32)
    nxt = torch.tensor([1, 2, 3, 3, 0, 3], dtype=torch.int32)
    acc = torch.tensor([0, 0, 0, 1], dtype=torch.uint8)
    aut = wl.Automaton(V=V, S=4, start=0, row_ptr=rp, tok=tok, next=nxt, accepting=acc)
    W[31] = W[30]
    W[32] = W[30]  # three identical rows -> -log 3, lowest id
    rm = [4, 2, 0, 5]
    tk, lp, lse, dn, st, gap = oracle.head_step(aut, hid, W, H, [0, 1, 2, 3], row_map=rm)
    x = f64(hid) @ f64(W).T
    assert tk[0] == 5 and lp[0] == 0.0 and abs(lse[0] - x[4, 5]) < 1e-12 and st[0] == 1 and gap[0] == math.inf
    d = abs(x[2, 7] - x[2, 20])
    assert tk[1] == (7 if x[2, 7] >= x[2, 20] else 20)
    assert abs(lp[1] + math.log1p(math.exp(-d))) < 1e-12 and abs(gap[1] - d) < 1e-12
    assert tk[2] == 30 and abs(lp[2] + math.log(3.0)) < 1e-12 and st[2] == 3 and dn[2] == 1 and gap[2] == 0.0
    assert tk[3] == -1 and lp[3] == 0.0 and dn[3] == 1 and st[3] == 3  # accepted rows never advance
    # row independence: each slot alone gives the same answer
    for i in range(3):
        t1, l1, e1, d1, s1, g1 = oracle.head_step(aut, hid, W, H, [i], row_map=[rm[i]])
        assert t1[0] == tk[i] and l1[0] == lp[i] and e1[0] == lse[i] and s1[0] == st[i]


def test_poisoned_complement_and_nan(oracle):
    V, H = 128, 32
    aut = wl.make_random_dfa(4, V, 6, 0.2, 0.2)
    hid = wl.make_hidden(4, 0, 5, H)
    W = wl.make_head(4, V, H, 2.0)
    state = [0, 0, 0, 0, 0]
    base = oracle.head_step(aut, hid, W, H, state)
    lo, hi = int(aut.row_ptr[0]), int(aut.row_ptr[1])
    allowed = set(int(t) for t in aut.tok[lo:hi])
    W2 = W.clone()
    for t in range(V):
        if t not in allowed:
            W2[t] = float("nan") if t % 2 else 1e30
    got = oracle.head_step(aut, hid, W2, H, state)
    for a, b in zip(base, got):
        assert np.array_equal(a, b)
    # an allowed NaN logit is read as -inf: same as removing the token's contribution
    t0 = sorted(allowed)[0]
    W3 = W.clone()
    W3[t0] = float("nan")
    tk, lp, lse, dn, st, gap = oracle.head_step(aut, hid, W3, H, state)
    x = f64(hid) @ f64(W).T
    rest = sorted(allowed - {t0})
    for r in range(5):
        xs = x[r, rest]
        assert tk[r] == rest[int(np.argmax(xs))]
        assert abs(lse[r] - (xs.max() + math.log(np.exp(xs - xs.max()).sum()))) < 1e-12


@pytest.mark.parametrize("kind", ["dfa", "trie"])
def test_head_loop_reduces_to_loop_on_library_matmul(oracle, kind):
    """O7 against the pinned O4 (oracle.decode_loop) fed with logits from a library matmul:
    exact-arithmetic inputs make the fp32 logits equal to the real dot products."""
    V, H, B, steps = 400, 96, 23, 6
    if kind == "dfa":
        aut = wl.make_random_dfa(21, V, 9, 0.2, 0.25)
    else:
        aut = wl.make_trie(V, wl.draw_labels(21, V, 12, 1, 4))
    W = wl.make_head(21, V, H, 2.0, exact=True, ld=H + 8)
    hs = [wl.make_hidden(21, k, B, H, exact=True) for k in range(steps)]
    logits = []
    for h in hs:
        x = f64(h[:, :H]) @ f64(W[:, :H]).T
        x32 = x.astype(np.float32)
        assert np.array_equal(x32.astype(np.float64), x)
        logits.append(x32)
    want = oracle.decode_loop(aut, logits)
    got = oracle.head_decode_loop(aut, hs, W, H)
    for k in ("tokens", "len", "final_state", "done", "n_active_hist"):
        assert np.array_equal(got[k], want[k]), k
    assert np.allclose(got["sum_logprob"], want["sum_logprob"], rtol=0, atol=1e-11)
    assert want["n_active_hist"][0] == B and want["len"].max() > 1  # the loop really iterates
