"""Pins for O11 (oracle/oracle_types.py): the EOS / longest-match variant of "when is a row
finished" (PAPER.md L61 option sets, L226 decoding rule left open).

Pinned against things other than the builder itself: a CSR written out by hand for the option set
{"a", "a b"}, the language enumerated by DFS over the CSR, decoding worked out by hand from four
logits, and the leaf-per-label trie of workloads.make_trie on prefix-free sets.  A plausible
mistake (eos edge missing from an inner may-stop state, several sinks, an accepting inner state,
a label's last edge going to the sink without eos, wrong numbering) fails one of them.
"""
import itertools
import math

import numpy as np
import pytest
import torch

import workloads as wl


def language(aut, max_len=64):
    rp, tk, nx, ac = aut.row_ptr, aut.tok, aut.next, aut.accepting
    out = []

    def dfs(s, prefix):
        assert len(prefix) <= max_len
        if ac[s]:
            out.append(tuple(prefix))
            return  # first accepting state ends the row (G4)
        assert rp[s + 1] > rp[s], "dead state"
        for j in range(int(rp[s]), int(rp[s + 1])):
            dfs(int(nx[j]), prefix + [int(tk[j])])

    dfs(aut.start, [])
    return out


def test_hand_case_a_and_a_b(oracle):
    """labels "a" = [5] and "a b" = [5, 6], eos = 2, V = 8.  By hand: 0 root, 1 after a (may stop),
    2 after a b (may stop), 3 the accepting sink."""
    aut = oracle.trie_eos(8, [[5], [5, 6]], eos=2)
    assert aut.S == 4 and aut.start == 0
    assert aut.row_ptr.tolist() == [0, 1, 3, 4, 4]
    assert aut.tok.tolist() == [5, 2, 6, 2]
    assert aut.next.tolist() == [1, 3, 2, 3]
    assert aut.accepting.tolist() == [0, 0, 0, 1]
    assert oracle.validate(aut) == 0
    # the order of the labels does not change the language, only the numbering of inner states
    assert sorted(language(oracle.trie_eos(8, [[5, 6], [5]], eos=2))) == [(5, 2), (5, 6, 2)]


def test_hand_case_decoding_is_the_models_choice_token_by_token(oracle):
    """Row 0 prefers eos after "a" (stops: label "a"), row 1 prefers b (goes on: "a b" then eos is
    forced), row 2 ties eos (id 2) with b (id 6): lowest id wins, so it stops."""
    aut = oracle.trie_eos(8, [[5], [5, 6]], eos=2)
    x0 = torch.full((3, 8), 9.0)  # step 0: only token 5 is allowed whatever the logits say
    x1 = torch.zeros(3, 8)
    x1[0, 2], x1[0, 6] = 1.5, -0.5
    x1[1, 2], x1[1, 6] = -1.0, 2.0
    x1[2, 2], x1[2, 6] = 0.25, 0.25
    x1[:, 7] = 50.0  # disallowed everywhere
    x2 = torch.full((3, 8), -3.0)
    res = oracle.decode_loop(aut, [x0, x1, x2, x2])
    assert res["tokens"].tolist() == [[5, 2, -1, -1], [5, 6, 2, -1], [5, 2, -1, -1]]
    assert res["len"].tolist() == [2, 3, 2] and res["done"].tolist() == [1, 1, 1]
    assert res["final_state"].tolist() == [3, 3, 3]  # one sink
    want = [-math.log1p(math.exp(-2.0)), -math.log1p(math.exp(-3.0)), -math.log(2.0)]
    np.testing.assert_allclose(res["sum_logprob"], want, rtol=0, atol=1e-12)


@pytest.mark.parametrize("seed,K", [(1, 5), (2, 12), (3, 40)])
def test_language_is_labels_plus_eos(oracle, seed, K):
    V, eos = 64, 63
    rng = np.random.default_rng(seed)
    labels = set()
    while len(labels) < K:
        base = tuple(int(t) for t in rng.integers(0, V - 1, size=int(rng.integers(1, 4))))
        labels.add(base)
        if rng.random() < 0.6:  # force prefix relations: the case G5 is about
            labels.add(base + tuple(int(t) for t in rng.integers(0, V - 1, size=int(rng.integers(1, 3)))))
    labels = [list(l) for l in sorted(labels)]
    rng.shuffle(labels)
    assert any(a != b and a == b[: len(a)] for a in labels for b in labels), "no prefix pair drawn"
    aut = oracle.trie_eos(V, labels, eos)
    lang = language(aut)
    assert len(lang) == len(set(lang)) == len(labels)
    assert set(lang) == {tuple(l) + (eos,) for l in labels}
    assert oracle.validate(aut) == 0
    # exactly one accepting state; it is the last one and a sink; eos leads nowhere else
    assert aut.accepting.tolist() == [0] * (aut.S - 1) + [1]
    assert aut.row_ptr[aut.S] == aut.row_ptr[aut.S - 1]
    assert set(aut.next[aut.tok == eos].tolist()) == {aut.S - 1}
    assert not np.any((aut.next == aut.S - 1) & (aut.tok != eos))
    # the may-stop states are exactly the states reached by a whole label
    rp, tk, nx = aut.row_ptr, aut.tok, aut.next
    for lab in labels:
        s = 0
        for t in lab:
            row = tk[rp[s]:rp[s + 1]].tolist()
            s = int(nx[rp[s] + row.index(t)])
        assert eos in tk[rp[s]:rp[s + 1]].tolist()
    n_may_stop = sum(1 for s in range(aut.S) if eos in tk[rp[s]:rp[s + 1]].tolist())
    assert n_may_stop == len(labels)


def test_numbering_is_insertion_order_with_the_sink_last(oracle):
    aut = oracle.trie_eos(100, [[7, 8, 9], [7, 3], [1]], eos=0)
    # 0 root, 1 = (7), 2 = (7,8), 3 = (7,8,9), 4 = (7,3), 5 = (1), 6 = sink
    assert aut.S == 7
    rows = [dict(zip(aut.tok[aut.row_ptr[s]:aut.row_ptr[s + 1]].tolist(),
                     aut.next[aut.row_ptr[s]:aut.row_ptr[s + 1]].tolist())) for s in range(aut.S)]
    assert rows == [{1: 5, 7: 1}, {3: 4, 8: 2}, {9: 3}, {0: 6}, {0: 6}, {0: 6}, {}]


def test_rejections(oracle):
    for labels, eos in (([[4], [4]], 2), ([[4], []], 2), ([[4, 2]], 2), ([[4]], 8), ([[4]], -1), ([[9]], 2)):
        with pytest.raises(ValueError):
            oracle.trie_eos(8, labels, eos)
    with pytest.raises(ValueError):  # without eos a prefix pair makes the longer string unreachable (G5)
        oracle.language_dfa(8, [[4], [4, 5]])


@pytest.mark.parametrize("name", ["c1", "c2"])
def test_prefix_free_sets_same_language_as_the_leaf_per_label_trie(oracle, name):
    cfg = wl.scaled(wl.CONFIGS[name], V=5000)
    trie = wl.build_automaton(cfg)
    plain = oracle.language_dfa(cfg.V, trie.labels)
    assert sorted(language(plain)) == sorted(tuple(l) for l in trie.labels) == sorted(language(trie))
    with_eos = oracle.trie_eos(cfg.V, trie.labels, eos=cfg.V - 1) if all(cfg.V - 1 not in l for l in trie.labels) else None
    if with_eos is not None:
        assert sorted(language(with_eos)) == sorted(tuple(l) + (cfg.V - 1,) for l in trie.labels)
        assert with_eos.S == trie.S + 1  # every leaf became a may-stop state, plus the sink


def test_list_language_written_out(oracle):
    labels, open_, sep, close = [[5], [5, 6]], [1], [2], [3]
    got = oracle.list_language(labels, open_, sep, close, 1, 2, eos=0)
    want = set()
    for c in (1, 2):
        for items in itertools.product(labels, repeat=c):
            seq = list(open_)
            for i, it in enumerate(items):
                seq += (list(sep) if i else []) + list(it)
            want.add(tuple(seq + close + [0]))
    assert len(got) == len(set(got)) and set(got) == want
    aut = oracle.language_dfa(8, got)
    assert sorted(language(aut)) == sorted(want) and oracle.validate(aut) == 0
    assert oracle.list_language([[4]], [], [], [9], 0, 1) == [(9,), (4, 9)]
