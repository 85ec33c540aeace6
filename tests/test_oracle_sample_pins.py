"""Pins for the oracle's sampled step (oracle_cd.c O10) against things other
than itself: libm's log, the Gumbel distribution's closed-form CDF and moments, the softmax
probabilities the Gumbel-max rule must reproduce (chi-square), torch log_softmax for the
reported log-probability, the greedy oracle O2 in the limit T -> 0, and a python-list
replay of the loop."""
import math

import numpy as np
import pytest
import torch

import workloads as wl


def test_det_logf_against_libm(oracle):
    xs = np.concatenate([np.exp(np.linspace(-17.0, 4.0, 4001)), 1.0 + np.linspace(-2e-3, 2e-3, 801),
                         [2.0**-24, 1.0 - 2.0**-24, 16.7, 0.5, 2.0, math.sqrt(0.5), math.sqrt(2.0)]]).astype(np.float32)
    for x in xs:
        ref = math.log(float(x))
        got = oracle.det_logf(float(x))
        assert abs(got - ref) <= 3e-7 * abs(ref) + 1e-9, (float(x), got, ref)
    assert oracle.det_logf(1.0) == 0.0


def test_gumbel_noise_distribution(oracle):
    g = np.array([oracle.gumbel(12345, r, 3, t) for r in range(40) for t in range(2500)])
    assert abs(g.mean() - 0.5772156649) < 0.02 and abs(g.var() - math.pi**2 / 6) < 0.05
    u = np.exp(-np.exp(-g))  # closed-form CDF: must be uniform
    hist, _ = np.histogram(u, bins=20, range=(0.0, 1.0))
    chi2 = float(((hist - g.size / 20) ** 2 / (g.size / 20)).sum())
    assert chi2 < 50.0, chi2  # 19 degrees of freedom: P(chi2 > 50) ~ 1e-4
    # counter-based: a pure function of its arguments, sensitive to each of them
    assert oracle.gumbel(1, 2, 3, 4) == oracle.gumbel(1, 2, 3, 4)
    base = oracle.gumbel(1, 2, 3, 4)
    assert all(oracle.gumbel(*a) != base for a in [(2, 2, 3, 4), (1, 3, 3, 4), (1, 2, 4, 4), (1, 2, 3, 5),
                                                   (1 + (1 << 32), 2, 3, 4)])


def small_automaton(V, allowed):
    rp = torch.tensor([0, len(allowed), len(allowed)], dtype=torch.int64)
    tok = torch.tensor(sorted(allowed), dtype=torch.int32)
    nxt = torch.ones(len(allowed), dtype=torch.int32)
    acc = torch.tensor([0, 1], dtype=torch.uint8)
    return wl.Automaton(V=V, S=2, start=0, row_ptr=rp, tok=tok, next=nxt, accepting=acc)


@pytest.mark.parametrize("T", [1.0, 0.5, 2.5])
def test_sampled_tokens_follow_the_masked_softmax(oracle, T):
    V, n = 64, 40000
    allowed = [3, 10, 11, 40, 63]
    aut = small_automaton(V, allowed)
    x = torch.full((1, V), 50.0)  # disallowed logits are huge: the mask must hide them
    x[0, allowed] = torch.tensor([0.0, 1.0, -1.0, 2.0, 0.5])
    tok, lp, lse, dn, st = oracle.sample_step(aut, x.expand(n, V).contiguous(), [0] * n, T, seed=77, step=1)
    y = (x[0, allowed].double() / T)
    p = torch.softmax(y, dim=0).numpy()
    counts = np.array([(tok == t).sum() for t in allowed])
    assert counts.sum() == n  # only allowed tokens are ever drawn
    chi2 = float(((counts - n * p) ** 2 / (n * p)).sum())
    assert chi2 < 30.0, (chi2, counts, n * p)  # 4 degrees of freedom: P(chi2 > 30) ~ 5e-6
    # reported log-probability = library log_softmax of the tempered logits at the drawn token
    y32 = (x[0, allowed].float() * np.float32(1.0 / np.float32(T))).double()
    ls = torch.log_softmax(y32, dim=0).numpy()
    for i in range(0, n, 997):
        k = allowed.index(int(tok[i]))
        assert abs(lp[i] - ls[k]) < 1e-12 and abs(lse[i] - float(torch.logsumexp(y32, 0))) < 1e-12
    assert (dn == 1).all() and (st == 1).all()


def test_low_temperature_is_greedy_and_identity_of_the_noise(oracle):
    V, S, n = 500, 9, 60
    aut = wl.make_random_dfa(41, V, S, 0.2, 0.2)
    x = wl.make_logits(41, 0, n, V, 2.0, torch.float32)
    acc = np.asarray(aut.accepting)
    live = [s for s in range(S) if not acc[s]]
    states = [live[i % len(live)] for i in range(n)]
    g_tok, _, _, g_dn, g_st = oracle.step(aut, x, states)
    tok, lp, lse, dn, st = oracle.sample_step(aut, x, states, 1e-4, seed=5)  # gaps / T >> noise
    assert np.array_equal(tok, g_tok) and np.array_equal(st, g_st) and np.array_equal(dn, g_dn)
    # the noise belongs to the ORIGINAL row id: permuting the slots permutes the results
    perm = np.random.default_rng(0).permutation(n)
    a = oracle.sample_step(aut, x, states, 1.0, seed=9, step=2)
    b = oracle.sample_step(aut, x, [states[i] for i in perm], 1.0, seed=9, step=2, row_map=perm.tolist())
    assert np.array_equal(b[0], a[0][perm]) and np.array_equal(b[1], a[1][perm])
    # other seed / step: other draws (with overwhelming probability not all equal)
    assert not np.array_equal(oracle.sample_step(aut, x, states, 1.0, seed=10, step=2)[0], a[0])
    assert not np.array_equal(oracle.sample_step(aut, x, states, 1.0, seed=9, step=3)[0], a[0])
    # every sampled token is allowed in its state; log-probs are <= 0 and <= the greedy token's
    rp, tk = np.asarray(aut.row_ptr), np.asarray(aut.tok)
    for i in range(n):
        assert a[0][i] in tk[rp[states[i]]:rp[states[i] + 1]]
    assert (a[1] <= 1e-12).all()


def test_sampled_loop_replays_as_steps_and_list_filter(oracle):
    V, S, B, steps = 300, 8, 40, 6
    aut = wl.make_random_dfa(43, V, S, 0.2, 0.2)
    logits = [wl.make_logits(43, k, B, V, 2.0, torch.float32) for k in range(steps)]
    got = oracle.sample_decode_loop(aut, logits, 0.8, seed=3, step_base=5)
    ids, st = list(range(B)), [aut.start] * B
    want_tok = -np.ones((B, steps), np.int32)
    want_len = np.zeros(B, np.int32)
    want_slp = np.zeros(B)
    for k in range(steps):
        if not ids:
            break
        tok, lp, lse, dn, ns = oracle.sample_step(aut, logits[k], st, 0.8, seed=3, step=5 + k, row_map=ids)
        for i, r in enumerate(ids):
            want_tok[r, k] = tok[i]
            want_len[r] = k + 1
            want_slp[r] += lp[i]
        keep = [i for i in range(len(ids)) if not dn[i]]
        ids, st = [ids[i] for i in keep], [int(ns[i]) for i in keep]
    assert np.array_equal(got["tokens"], want_tok) and np.array_equal(got["len"], want_len)
    assert np.allclose(got["sum_logprob"], want_slp, rtol=0, atol=1e-12)
    assert want_len.max() > 1


# ---------------------------------------------------------------- the integer side of the generator, from outside
# MurmurHash3_x86_32 of the EMPTY key is fmix32(seed) (no blocks, no tail, length 0), so the reference vectors
# that every murmur3 port is verified with pin the finalizer itself:
#   murmur3_32("", seed 0) = 0x00000000, ("", seed 1) = 0x514E28B7, ("", seed 0xFFFFFFFF) = 0x81F16F39
MURMUR3_EMPTY_KEY = [(0x00000000, 0x00000000), (0x00000001, 0x514E28B7), (0xFFFFFFFF, 0x81F16F39)]


def test_fmix32_against_murmur3_published_vectors(oracle):
    for seed, want in MURMUR3_EMPTY_KEY:
        assert oracle.fmix32(seed) == want, (hex(seed), hex(oracle.fmix32(seed)), hex(want))
    # a bijection on 32-bit words (xorshifts and odd multipliers): no two of many inputs collide
    xs = np.random.default_rng(5).integers(0, 2**32, size=20000, dtype=np.uint64)
    assert len({oracle.fmix32(int(x)) for x in set(xs.tolist())}) == len(set(xs.tolist()))
    # avalanche: flipping one input bit flips about half of the output bits
    flips = [bin(oracle.fmix32(int(x)) ^ oracle.fmix32(int(x) ^ (1 << b))).count("1") for x in xs[:300] for b in range(32)]
    assert 15.0 < np.mean(flips) < 17.0 and min(flips) >= 1


AXES = ["seed_lo", "seed_hi", "row", "step", "tok"]


def _g(oracle, seed_lo=0x9ABCDEF0, seed_hi=0x12345678, row=1234, step=7, tok=4321):
    return oracle.gumbel((seed_hi << 32) | seed_lo, row, step, tok)


@pytest.mark.parametrize("axis", AXES)
def test_noise_depends_on_every_input_varied_alone(oracle, axis):
    """A generator that dropped (or merely truncated) one of its five inputs would return a constant, or a short
    cycle, along that axis.  4096 consecutive values of the axis and 4096 values with only a high bit pattern
    changing: all distinct uniforms, uniformly spread, and neighbours uncorrelated."""
    n = 4096
    for vals in (range(n), [(i * 0x00100001) & 0xFFFFFFFF for i in range(n)], [(i << 20) & 0xFFFFFFFF for i in range(n)]):
        g = np.array([_g(oracle, **{axis: int(v)}) for v in vals])
        u = np.exp(-np.exp(-g))
        assert len(np.unique(g)) > 0.995 * n, (axis, len(np.unique(g)))  # (24-bit uniforms: a few birthdays at most)
        hist, _ = np.histogram(u, bins=16, range=(0.0, 1.0))
        chi2 = float(((hist - n / 16) ** 2 / (n / 16)).sum())
        assert chi2 < 45.0, (axis, chi2)  # 15 degrees of freedom: P(chi2 > 45) ~ 8e-5
        c = np.corrcoef(u[:-1], u[1:])[0, 1]
        assert abs(c) < 0.08, (axis, c)  # 5 sigma of 1 / sqrt(n)


def test_noise_streams_of_different_inputs_are_unrelated(oracle):
    """Two axes never alias: the stream over tokens of (row r, step k) is uncorrelated with the one of (row r + 1,
    step k), (row r, step k + 1), of the swapped pair (row k, step r), and of a seed differing in its high or low
    word only."""
    n = 4096
    def stream(**kw):
        return np.exp(-np.exp(-np.array([_g(oracle, tok=t, **kw) for t in range(n)])))
    base = stream(row=10, step=3)
    others = [stream(row=11, step=3), stream(row=10, step=4), stream(row=3, step=10),
              stream(row=10, step=3, seed_hi=0x12345679), stream(row=10, step=3, seed_lo=0x9ABCDEF1)]
    for o in others:
        assert not np.array_equal(o, base)
        assert abs(np.corrcoef(base, o)[0, 1]) < 0.08
