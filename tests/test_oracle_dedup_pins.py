"""Pins for the oracle's early deduplication / join / cascade filter (oracle_cd.c O8, O9;
PAPER.md section 2.4, L150 and L156) against things other than itself: numpy's library
`unique` (re-ordered by first index), a python dict, the algebraic identities of
DISTINCT + LEFT JOIN, and list comprehensions."""
import numpy as np
import pytest

import workloads as wl


@pytest.mark.parametrize("N,nv,skew", [(1, 1, False), (50, 1, False), (1000, 37, False), (5000, 900, True),
                                       (300, 100000, False)])
def test_dedup_against_library_unique_and_dict(oracle, N, nv, skew):
    keys = wl.make_keys(3, N, nv, skew=skew).numpy()
    rep, dr = oracle.dedup(keys)
    # numpy: sorted unique values with first indices and inverse; re-order by first occurrence
    u, first_idx, inv = np.unique(keys, return_index=True, return_inverse=True)
    order = np.argsort(first_idx)
    pos = np.empty_like(order)
    pos[order] = np.arange(order.size)
    assert np.array_equal(dr, first_idx[order])
    assert np.array_equal(rep, pos[inv])
    # python dict, insertion ordered
    seen = {}
    for i, k in enumerate(keys.tolist()):
        seen.setdefault(k, (len(seen), i))
    assert [seen[k][0] for k in keys.tolist()] == rep.tolist()
    assert [v[1] for v in seen.values()] == dr.tolist()
    # identities: the join key reproduces every row's value; first rows map to themselves
    assert np.array_equal(keys[dr[rep]], keys)
    assert np.array_equal(rep[dr], np.arange(dr.size))
    assert np.all(np.diff(dr) > 0)


def test_dedup_extreme_keys(oracle):
    keys = np.array([np.iinfo(np.int64).min, 0, -1, np.iinfo(np.int64).max, np.iinfo(np.int64).min, -1, 7],
                    dtype=np.int64)
    rep, dr = oracle.dedup(keys)
    assert rep.tolist() == [0, 1, 2, 3, 0, 2, 4] and dr.tolist() == [0, 1, 2, 3, 6]
    rep, dr = oracle.dedup(np.zeros(0, np.int64))
    assert rep.size == 0 and dr.size == 0


def test_join_is_a_gather_and_commutes_with_decoding(oracle):
    """Decoding the distinct rows and joining back equals decoding every row, when rows with the
    same value carry the same logits (the premise of the optimisation)."""
    V, nv, N, steps = 300, 9, 60, 5
    aut = wl.make_random_dfa(31, V, 8, 0.2, 0.2)
    keys = wl.make_keys(31, N, nv).numpy()
    rep, dr = oracle.dedup(keys)
    per_value = [wl.make_logits(31, k, len(dr), V, 2.0, __import__("torch").float32) for k in range(steps)]
    full = [x[rep.astype(np.int64)] for x in per_value]  # row i sees the logits of its value
    res_d = oracle.decode_loop(aut, per_value)
    res_f = oracle.decode_loop(aut, full)
    joined = oracle.join_results(rep, res_d)
    for k in ("tokens", "len", "final_state", "sum_logprob", "done"):
        assert np.array_equal(joined[k], res_f[k]), k
        assert np.array_equal(joined[k], np.asarray(res_d[k])[rep]), k  # numpy fancy indexing


def test_filter_rows_is_a_list_filter(oracle):
    rng = np.random.default_rng(5)
    S, N = 11, 500
    fs = rng.integers(0, S, N).astype(np.int32)
    dn = (rng.random(N) < 0.7).astype(np.uint8)
    sat = (rng.random(S) < 0.4).astype(np.uint8)
    ids = rng.permutation(N).astype(np.int32)
    want = [i for i in range(N) if dn[i] and sat[fs[i]]]
    assert oracle.filter_rows(fs, dn, sat).tolist() == want
    assert oracle.filter_rows(fs, dn, sat, row_ids=ids).tolist() == [int(ids[i]) for i in want]
    assert oracle.filter_rows(fs, np.zeros(N, np.uint8), sat).size == 0
    # chaining two predicates = conjunction
    fs2 = rng.integers(0, S, N).astype(np.int32)
    first = oracle.filter_rows(fs, dn, sat)
    second = oracle.filter_rows(fs2[first], np.ones(first.size, np.uint8), sat, row_ids=first)
    assert second.tolist() == [i for i in want if sat[fs2[i]]]
