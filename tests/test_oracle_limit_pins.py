"""Pins for the oracle's LIMIT early exit (oracle_cd.c O5; section 2.4
"Early Exiting", L152-L154) against things other than itself.

The limited loop is fully determined by the unlimited one: rows are independent
(PAPER.md L106), so until the exit step every row does what it does without a
limit, and the exit step is the first step after which the number of rows that
finished in a satisfying state reaches the limit.  The expectation is rebuilt
here from the UNLIMITED result with python lists (finish step per row,
cumulative count, truncation, replay through a dict) -- a different formulation
from the C loop, which counts while it runs.
"""
import numpy as np
import pytest
import torch

import workloads as wl


def expected_from_unlimited(aut, full, satisfying, limit, satisfied0, max_steps):
    rp, tk, nx = (np.asarray(a) for a in (aut.row_ptr, aut.tok, aut.next))
    delta = {}
    for s in range(aut.S):
        for j in range(int(rp[s]), int(rp[s + 1])):
            delta[(s, int(tk[j]))] = int(nx[j])
    B = full["len"].shape[0]
    want = {k: np.array(v, copy=True) for k, v in full.items() if k != "n_active_hist"}
    if satisfied0 >= limit:  # nothing runs
        want["tokens"][:] = -1
        want["len"][:] = 0
        want["final_state"][:] = aut.start
        want["sum_logprob"][:] = 0.0
        want["done"][:] = 1 if np.asarray(aut.accepting)[aut.start] else 0
        return want, satisfied0, -1
    # rows finishing (accepted) at step k in a satisfying state
    per_step = [0] * max_steps
    for r in range(B):
        if full["done"][r] and full["len"][r] > 0 and satisfying[full["final_state"][r]]:
            per_step[full["len"][r] - 1] += 1
    cum, exit_step = satisfied0, None
    for k in range(max_steps):
        cum += per_step[k]
        if cum >= limit:
            exit_step = k
            break
    if exit_step is None:
        return want, cum, None
    keep = exit_step + 1  # tokens a cancelled row keeps
    for r in range(B):
        if full["len"][r] > keep:
            want["tokens"][r, keep:] = -1
            want["len"][r] = keep
            want["done"][r] = 0
            s = aut.start
            for k in range(keep):
                s = delta[(s, int(full["tokens"][r, k]))]
            want["final_state"][r] = s
            want["sum_logprob"][r] = np.nan  # checked separately (prefix sum of per-step log-probs)
    return want, cum, exit_step


def run_case(oracle, aut, logits, max_steps, satisfying, limit, satisfied0=0):
    full = oracle.decode_loop(aut, logits, max_steps=max_steps)
    got = oracle.decode_loop(aut, logits, max_steps=max_steps, satisfying=satisfying, limit=limit,
                             satisfied=satisfied0)
    want, cum, exit_step = expected_from_unlimited(aut, full, satisfying, limit, satisfied0, max_steps)
    for k in ("tokens", "len", "final_state", "done"):
        assert np.array_equal(got[k], want[k]), k
    assert got["satisfied"] == cum
    same = ~np.isnan(want["sum_logprob"])
    assert np.array_equal(got["sum_logprob"][same], want["sum_logprob"][same])
    # a cancelled row's sum is a prefix of its unlimited history: never below the full sum's
    # magnitude (every term is <= 0) and exactly the sum of step() log-probs along the prefix
    cancelled = np.nonzero(~same)[0]
    for r in cancelled[:20]:
        s, acc = aut.start, 0.0
        for k in range(int(got["len"][r])):
            _, lp, _, _, st = oracle.step(aut, logits[k][r:r + 1], [s])
            acc += float(lp[0])
            s = int(st[0])
        assert abs(acc - got["sum_logprob"][r]) <= 1e-12 * max(1.0, abs(acc))
        assert got["sum_logprob"][r] >= full["sum_logprob"][r] - 1e-12
    return got, full, exit_step


def test_limit_on_config_c0_by_hand(oracle):
    """BASELINE.json configs[0]: step 0 picks 42 ('false', done) or 17; LIMIT 1 on `= FALSE`
    stops after step 0 as soon as any row said false: the rows that chose 17 keep one token."""
    cfg = wl.CONFIGS["c0"]
    aut = wl.build_automaton(cfg)
    logits = wl.build_step_logits(cfg, aut, device="cpu")
    x0 = logits[0]
    first = [17 if float(x0[r, 17]) >= float(x0[r, 42]) else 42 for r in range(cfg.B)]
    assert 42 in first and 17 in first, "seeded c0 logits must exercise both branches"
    leaf_false = int(aut.leaf_of_label[[tuple(l) for l in aut.labels].index((42,))])
    sat = np.zeros(aut.S, np.uint8)
    sat[leaf_false] = 1
    got = oracle.decode_loop(aut, logits, satisfying=sat, limit=1)
    assert got["satisfied"] == first.count(42)
    for r in range(cfg.B):
        assert got["len"][r] == 1 and got["tokens"][r, 0] == first[r]
        assert got["done"][r] == (1 if first[r] == 42 else 0)
    # LIMIT larger than the table has: nothing is cancelled
    got2 = oracle.decode_loop(aut, logits, satisfying=sat, limit=cfg.B + 1)
    full = oracle.decode_loop(aut, logits)
    for k in ("tokens", "len", "final_state", "done", "sum_logprob"):
        assert np.array_equal(got2[k], full[k])
    assert got2["satisfied"] == first.count(42)


@pytest.mark.parametrize("limit", [1, 5, 40, 10**6])
@pytest.mark.parametrize("satisfied0", [0, 3])
def test_limit_derived_from_unlimited_loop_random_dfa(oracle, limit, satisfied0):
    cfg = wl.scaled(wl.CONFIGS["c3"], V=2048, B=120, S=40, max_steps=12)
    aut = wl.build_automaton(cfg)
    logits = wl.build_step_logits(cfg, aut, device="cpu")
    acc = np.asarray(aut.accepting)
    sat = (acc * (np.arange(aut.S) % 2 == 0)).astype(np.uint8)  # half of the accepting states satisfy
    assert sat.sum() > 0
    got, full, exit_step = run_case(oracle, aut, logits, cfg.max_steps, sat, limit, satisfied0)
    if limit == 10**6:
        assert exit_step is None and np.array_equal(got["len"], full["len"])
    if limit == 1 and satisfied0 == 3:
        assert int(got["len"].max()) == 0  # already satisfied at entry: no row takes a step


def test_limit_on_trie_labels(oracle):
    """`options` classifier with LIMIT: stop once 7 rows got label 3."""
    cfg = wl.scaled(wl.CONFIGS["c2"], V=5000, B=300, K=12)
    aut = wl.build_automaton(cfg)
    logits = wl.build_step_logits(cfg, aut, device="cpu")
    sat = np.zeros(aut.S, np.uint8)
    sat[int(aut.leaf_of_label[3])] = 1
    got, full, exit_step = run_case(oracle, aut, logits, cfg.max_steps, sat, 7)
    n_label3 = int((full["final_state"] == int(aut.leaf_of_label[3])).sum())
    if n_label3 >= 7:
        assert exit_step is not None and got["satisfied"] >= 7
        assert got["satisfied"] <= n_label3
    # counting across batches of the table: second call starts from the first call's count
    again = oracle.decode_loop(aut, logits, satisfying=sat, limit=7, satisfied=got["satisfied"])
    if got["satisfied"] >= 7:
        assert int(again["len"].max()) == 0 and again["satisfied"] == got["satisfied"]


def test_limit_without_satisfying_is_the_plain_loop(oracle):
    cfg = wl.scaled(wl.CONFIGS["c3"], V=1024, B=33, S=16, max_steps=6)
    aut = wl.build_automaton(cfg)
    logits = wl.build_step_logits(cfg, aut, device="cpu")
    a = oracle.decode_loop(aut, logits)
    b = oracle.decode_loop(aut, logits, satisfying=None, limit=0)
    for k in ("tokens", "len", "final_state", "done", "sum_logprob"):
        assert np.array_equal(a[k], b[k])
