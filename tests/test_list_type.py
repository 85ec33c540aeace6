"""Collection types with a quantifier (cd_build_list / cd_compile_list; section 2.3):
the automaton's language, enumerated by DFS over the CSR, must be exactly
{ open + sep.join(items) + close : min_items <= len(items) <= max_items, items from the labels },
written out here with itertools.  Host logic: runs without a GPU; one GPU test decodes through it."""
import itertools

import numpy as np
import pytest
import torch

import workloads as wl


@pytest.fixture(scope="module")
def cd():
    import paper_2606_31808_b200 as m

    m.lib()
    return m


def language(S, rp, tk, nx, ac, start=0, max_len=64):
    rp, tk, nx, ac = (np.asarray(x) for x in (rp, tk, nx, ac))
    out = set()

    def dfs(s, prefix):
        assert len(prefix) <= max_len
        if ac[s]:
            out.add(tuple(prefix))
            assert rp[s + 1] == rp[s]  # the accepting state is a sink: "first accept" ends the list
            return
        assert rp[s + 1] > rp[s]  # no dead state
        for j in range(int(rp[s]), int(rp[s + 1])):
            dfs(int(nx[j]), prefix + [int(tk[j])])

    dfs(start, [])
    return out


def expected(labels, open_, sep, close, lo, hi):
    out = set()
    for c in range(lo, hi + 1):
        for items in itertools.product(labels, repeat=c):
            seq = list(open_)
            for i, it in enumerate(items):
                if i:
                    seq += list(sep)
                seq += list(it)
            out.add(tuple(seq + list(close)))
    return out


CASES = [
    ([[5], [6, 7], [6, 8]], [1], [2], [3], 1, 2),
    ([[5], [6, 7], [6, 8]], [], [2], [3], 0, 3),
    ([[10, 11, 12], [10, 11, 13], [20]], [1, 1], [2, 9], [3, 4], 2, 2),
    ([[7]], [0], [], [9], 1, 1),
    ([[4], [5]], [1], [2], [3], 0, 1),
    ([[4, 4], [4, 5], [6]], [], [4], [9], 3, 4),  # sep token also starts labels: roots are fresh states
]


@pytest.mark.parametrize("labels,open_,sep,close,lo,hi", CASES)
def test_language_is_the_quantified_list(cd, oracle, labels, open_, sep, close, lo, hi):
    V = 32
    S, rp, tk, nx, ac = cd.build_list(V, labels, open_, sep, close, lo, hi)
    assert language(S, rp, tk, nx, ac) == expected(labels, open_, sep, close, lo, hi)
    assert int(ac.sum()) == 1
    aut = wl.Automaton(V=V, S=S, start=0, row_ptr=rp, tok=tk, next=nx, accepting=ac)
    assert oracle.validate(aut) == 0  # O1: sorted tokens, no dead state, ranges
    # deterministic: tokens strictly increasing inside every state
    for s in range(S):
        row = tk[int(rp[s]):int(rp[s + 1])].tolist()
        assert row == sorted(set(row))


@pytest.mark.parametrize("kw,msg", [
    (dict(labels=[[5], [5, 6]]), "prefix"),
    (dict(labels=[[5], [5]]), "duplicate"),
    (dict(sep=[3]), "same token"),
    (dict(close=[]), "close"),
    (dict(sep=[], hi=2), "sep"),
    (dict(lo=0, labels=[[3]]), "close starts like a label"),
    (dict(lo=3, hi=2), "min_items"),
    (dict(labels=[[99]]), "outside"),
])
def test_rejected_inputs(cd, kw, msg):
    a = dict(labels=[[5], [6]], open_=[1], sep=[2], close=[3], lo=1, hi=2)
    a.update(kw)
    with pytest.raises(cd.CdError) as e:
        cd.build_list(32, a["labels"], a["open_"], a["sep"], a["close"], a["lo"], a["hi"])
    assert e.value.code == 2 and msg in str(e.value)


@pytest.mark.gpu
def test_decoding_through_a_list_type(cd, oracle):
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    V, B = 4096, 200
    labels = wl.draw_labels(81, V, 12, 1, 3)
    open_, sep, close = [V - 1], [V - 2], [V - 3]
    labels = [l for l in labels if l[0] < V - 3]
    lo, hi = 1, 3
    S, rp, tk, nx, ac = cd.build_list(V, labels, open_, sep, close, lo, hi)
    aut = wl.Automaton(V=V, S=S, start=0, row_ptr=rp, tok=tk, next=nx, accepting=ac)
    dfa = cd.compile_list(V, labels, open_, sep, close, lo, hi, device="cuda:0")
    assert dfa.S == S and dfa.nnz == tk.numel()
    steps = 2 + hi * 4 + (hi - 1)
    logits = [wl.make_logits(81, k, B, V, 2.0, torch.bfloat16) for k in range(steps)]
    got = cd.decode_loop(dfa, [x.to("cuda:0") for x in logits])
    torch.cuda.synchronize()
    want = oracle.decode_loop(aut, logits)
    for k in ("tokens", "len", "final_state", "done"):
        assert np.array_equal(got[k].cpu().numpy(), want[k]), k
    assert want["done"].all()
    lang = expected(labels, open_, sep, close, lo, hi)
    for r in range(0, B, 7):
        assert tuple(want["tokens"][r, : want["len"][r]].tolist()) in lang
