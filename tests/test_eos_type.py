"""The EOS / longest-match variant of the option-set and list types (
cd_build_trie / cd_compile_trie / cd_build_list / cd_compile_list with eos >= 0).

Host logic (no GPU): the product's builder (csrc/cd_types.hpp) against the oracle's definition-level
builder (oracle/oracle_types.py, O11) -- the two are written independently and must produce the same
CSR, array for array (the state numbering is part of the documented interface), and the same
language.  GPU: decoding through the compiled automaton against the oracle loop on the ORACLE's
automaton, greedy and sampled."""
import numpy as np
import pytest
import torch

import workloads as wl
from test_oracle_eos_pins import language


@pytest.fixture(scope="module")
def cd():
    import paper_2606_31808_b200 as m

    m.lib()
    return m


def prefix_heavy_labels(seed, V, K, eos):
    rng = np.random.default_rng(seed)
    labels = set()
    while len(labels) < K:
        base = tuple(int(t) for t in rng.choice([t for t in range(V) if t != eos], size=int(rng.integers(1, 4))))
        labels.add(base)
        if rng.random() < 0.6:
            ext = tuple(int(t) for t in rng.choice([t for t in range(V) if t != eos], size=int(rng.integers(1, 3))))
            labels.add(base + ext)
    labels = [list(l) for l in sorted(labels)]
    rng.shuffle(labels)
    return labels


def same_csr(got, want):
    S, rp, tk, nx, ac = got
    assert S == want.S
    assert rp.numpy().tolist() == want.row_ptr.tolist()
    assert tk.numpy().tolist() == want.tok.tolist()
    assert nx.numpy().tolist() == want.next.tolist()
    assert ac.numpy().tolist() == want.accepting.tolist()


def test_hand_case_matches_the_oracle_array_for_array(cd, oracle):
    same_csr(cd.build_trie(8, [[5], [5, 6]], eos=2), oracle.trie_eos(8, [[5], [5, 6]], 2))
    S, rp, tk, nx, ac = cd.build_trie(8, [[5], [5, 6]], eos=2)
    assert (S, rp.tolist(), tk.tolist(), nx.tolist(), ac.tolist()) == (4, [0, 1, 3, 4, 4], [5, 2, 6, 2], [1, 3, 2, 3], [0, 0, 0, 1])


@pytest.mark.parametrize("seed,V,K", [(1, 40, 6), (2, 64, 20), (3, 500, 60), (4, 9, 5)])
def test_builder_equals_the_oracle_definition(cd, oracle, seed, V, K):
    eos = V - 1 if seed % 2 else 0
    labels = prefix_heavy_labels(seed, V, K, eos)
    same_csr(cd.build_trie(V, labels, eos=eos), oracle.trie_eos(V, labels, eos))


def test_without_eos_the_trie_is_the_leaf_per_label_trie(cd, oracle):
    for name in ("c0", "c1", "c2"):
        cfg = wl.scaled(wl.CONFIGS[name], V=min(wl.CONFIGS[name].V, 5000))
        aut = wl.build_automaton(cfg)
        same_csr(cd.build_trie(cfg.V, aut.labels, eos=-1), aut)
        assert cd.build_trie(cfg.V, aut.labels)[0] == aut.S  # eos defaults to "none"


@pytest.mark.parametrize("labels,eos,msg", [
    ([[4], [4]], 2, "duplicate"), ([[4], []], 2, "empty"), ([[4, 2]], 2, "eos"), ([[4]], 8, "eos"),
    ([[9]], 2, "outside"), ([[4], [4, 5]], -1, "prefix"), ([[4, 5], [4]], -1, "prefix"),
])
def test_rejections(cd, oracle, labels, eos, msg):
    with pytest.raises(cd.CdError) as e:
        cd.build_trie(8, labels, eos=eos)
    assert e.value.code == 2 and msg in str(e.value)
    if eos >= 0:  # the oracle's definition rejects the same sets
        with pytest.raises(ValueError):
            oracle.trie_eos(8, labels, eos)


LIST_CASES = [
    # labels, open, sep, close, lo, hi, eos
    ([[5], [5, 6]], [1], [2], [3], 1, 2, 0),            # "a" / "a b" as items: the item ends when sep / close follows
    ([[5], [5, 6], [5, 6, 7], [9]], [], [2], [3], 0, 3, 0),
    ([[10, 11], [10, 11, 12], [20]], [1, 1], [2, 9], [3, 4], 2, 2, 31),
    ([[7]], [0], [], [9], 1, 1, 5),
    ([[5], [6, 7], [6, 8]], [1], [2], [3], 1, 2, 0),    # prefix-free items with eos: only the ending changes
]


@pytest.mark.parametrize("labels,open_,sep,close,lo,hi,eos", LIST_CASES)
def test_list_language_with_eos(cd, oracle, labels, open_, sep, close, lo, hi, eos):
    V = 32
    S, rp, tk, nx, ac = cd.build_list(V, labels, open_, sep, close, lo, hi, eos=eos)
    aut = wl.Automaton(V=V, S=S, start=0, row_ptr=rp, tok=tk, next=nx, accepting=ac)
    want = oracle.list_language(labels, open_, sep, close, lo, hi, eos=eos)
    assert len(want) == len(set(want))  # these cases are unambiguous
    got = language(aut)
    assert len(got) == len(set(got)) and set(got) == set(want)
    assert oracle.validate(aut) == 0 and int(ac.sum()) == 1
    ref = oracle.language_dfa(V, want)  # the definition-level automaton of the same language
    assert set(language(ref)) == set(got)


@pytest.mark.parametrize("kw,msg", [
    (dict(labels=[[5], [5, 2]], sep=[2]), "continues"),      # sep[0] continues the longer label: ambiguous
    (dict(labels=[[5], [5, 3]], close=[3]), "continues"),    # close[0] does
    (dict(labels=[[5], [5]]), "duplicate"),
    (dict(labels=[[5, 0]]), "eos"),
    (dict(close=[3, 0]), "eos"),
    (dict(eos=99), "eos"),
])
def test_list_rejections_with_eos(cd, kw, msg):
    a = dict(labels=[[5], [6]], open_=[1], sep=[2], close=[3], lo=1, hi=2, eos=0)
    a.update(kw)
    with pytest.raises(cd.CdError) as e:
        cd.build_list(32, a["labels"], a["open_"], a["sep"], a["close"], a["lo"], a["hi"], eos=a["eos"])
    assert e.value.code == 2 and msg in str(e.value)


# ------------------------------------------------------------------ GPU: decode through the compiled types
def _loop_equal(got, want, tol=1e-5, final_state=True):
    keys = ("tokens", "len", "done") + (("final_state",) if final_state else ())
    for k in keys:
        assert np.array_equal(got[k].cpu().numpy(), want[k]), k
    g, r = got["sum_logprob"].cpu().numpy().astype(np.float64), want["sum_logprob"]
    assert np.all(np.abs(g - r) <= np.maximum(tol * (want["len"] + np.abs(r)), tol))


@pytest.mark.gpu
@pytest.mark.parametrize("mode", ["auto", "barrier", "per_step"])
@pytest.mark.parametrize("gather", [0, 2**30])
def test_decoding_option_sets_with_eos_greedy_and_sampled(cd, oracle, mode, gather):
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    V, B, eos = 50000, 600, 7
    labels = prefix_heavy_labels(11, V, 40, eos)
    assert any(a != b and a == b[: len(a)] for a in labels for b in labels)
    aut = oracle.trie_eos(V, labels, eos)  # the ORACLE's automaton
    dfa = cd.compile_trie(V, labels, device="cuda:0", eos=eos)
    assert (dfa.S, dfa.nnz) == (aut.S, aut.nnz)
    dfa.set_gather_max(gather)
    dfa.set_loop_mode({"auto": cd.LOOP_AUTO, "barrier": cd.LOOP_BARRIER, "per_step": cd.LOOP_PER_STEP}[mode])
    steps = max(len(l) for l in labels) + 1
    # bias eos a little so that rows stop at inner may-stop states as well as at the longest labels
    logits = [wl.make_logits(11, k, B, V, 2.0, torch.bfloat16, device="cuda:0", bias_tokens=[eos], bias=1.0)
              for k in range(steps)]
    host = [x.cpu() for x in logits]
    got = cd.decode_loop(dfa, logits)
    want = oracle.decode_loop(aut, host)
    _loop_equal(got, want)
    assert want["done"].all() and set(want["final_state"].tolist()) == {aut.S - 1}
    lab_set = {tuple(l) for l in labels}
    lens = set()
    for r in range(B):
        h = want["tokens"][r, : want["len"][r]].tolist()
        assert h[-1] == eos and tuple(h[:-1]) in lab_set
        lens.add(len(h))
    assert len(lens) > 1
    # rows that stopped at a label which is a proper prefix of another label: the case G5 is about
    inner = {tuple(a) for a in labels for b in labels if a != b and a == b[: len(a)]}
    assert any(tuple(want["tokens"][r, : want["len"][r] - 1].tolist()) in inner for r in range(B))
    # sampled
    dfa.set_sampling(0.9, seed=77)
    got_s = cd.decode_loop(dfa, logits)
    want_s = oracle.sample_decode_loop(aut, host, 0.9, seed=77)
    _loop_equal(got_s, want_s)
    dfa.close()


@pytest.mark.gpu
def test_decoding_a_list_type_with_eos(cd, oracle):
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    V, B, eos = 4096, 300, 0
    labels = [[50], [50, 51], [50, 51, 52], [60, 61], [70]]
    open_, sep, close = [V - 1], [V - 2], [V - 3]
    lo, hi = 1, 3
    dfa = cd.compile_list(V, labels, open_, sep, close, lo, hi, device="cuda:0", eos=eos)
    lang = oracle.list_language(labels, open_, sep, close, lo, hi, eos=eos)
    ref = oracle.language_dfa(V, lang)  # numbering differs from the product's: compare what is unique
    steps = 1 + hi * 3 + (hi - 1) + 2 + 1
    logits = [wl.make_logits(83, k, B, V, 2.0, torch.bfloat16, device="cuda:0") for k in range(steps)]
    got = cd.decode_loop(dfa, logits)
    want = oracle.decode_loop(ref, [x.cpu() for x in logits])
    _loop_equal(got, want, final_state=False)
    assert want["done"].all()
    lang = set(lang)
    for r in range(B):
        assert tuple(want["tokens"][r, : want["len"][r]].tolist()) in lang
    dfa.close()
