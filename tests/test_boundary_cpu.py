"""Boundary checks that need no GPU: the C-ABI library loads, exports every
symbol include/cd.h declares, and its host-side automaton validation returns
the codes SURVEY.md 8(c) O1 fixes (the same malformed automata are given to
the oracle's validator; the two share no code)."""
import os
import re

import numpy as np
import pytest
import torch

import paper_2606_31808_b200 as cd
from paper_2606_31808_b200 import binding

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _header_symbols():
    inc = os.path.join(ROOT, "include")  # cd.h: the decoding contract; cd_diag.h: measurement aids of the same library
    text = "".join(open(os.path.join(inc, f)).read() for f in sorted(os.listdir(inc)) if f.endswith(".h"))
    return sorted(set(re.findall(r"CD_API[^;(]*?\b(cd_\w+)\s*\(", text)))


def test_library_is_built_in_tree_and_loads():
    assert os.path.exists(cd.lib_path()), "run: python -m paper_2606_31808_b200.build"
    assert cd.lib() is not None


def test_every_declared_symbol_is_exported():
    syms = _header_symbols()
    assert len(syms) >= 12
    assert set(syms) == set(binding.SYMBOLS)
    L = cd.lib()
    for s in syms:
        assert getattr(L, s) is not None


def test_required_entry_points_named_by_north_star():
    for s in ("cd_compile_dfa", "cd_step", "cd_compact", "cd_decode_loop"):
        assert s in _header_symbols()


def _compile_rc(V, S, start, rp, tok, nxt, acc):
    try:
        d = cd.compile_dfa(V, S, start, rp, tok, nxt, acc)
        d.close()
        return 0
    except cd.CdError as e:
        return e.code


class A:
    pass


CASES = [
    # (name, V, S, start, row_ptr, tok, next, accepting, expected code; 0 = valid)
    ("ok", 16, 2, 0, [0, 2, 2], [1, 4], [1, 0], [0, 1], 0),
    ("unsorted", 16, 2, 0, [0, 2, 2], [4, 1], [1, 0], [0, 1], 2),
    ("duplicate", 16, 2, 0, [0, 2, 2], [4, 4], [1, 0], [0, 1], 2),
    ("tok_oob", 16, 2, 0, [0, 1, 1], [16], [1], [0, 1], 2),
    ("tok_neg", 16, 2, 0, [0, 1, 1], [-1], [1], [0, 1], 2),
    ("next_oob", 16, 2, 0, [0, 1, 1], [3], [2], [0, 1], 2),
    ("start_oob", 16, 2, 2, [0, 1, 1], [3], [1], [0, 1], 2),
    ("rowptr_decreasing", 16, 2, 0, [0, 2, 1], [3, 4], [1, 1], [0, 1], 2),
    ("rowptr_nonzero", 16, 2, 0, [1, 2, 2], [3, 4], [1, 1], [0, 1], 2),
    ("dead_state", 16, 2, 0, [0, 1, 1], [3], [1], [0, 0], 3),
    ("accepting_leaf", 16, 2, 0, [0, 1, 1], [3], [1], [0, 1], 0),
]


@pytest.mark.parametrize("case", CASES, ids=[c[0] for c in CASES])
def test_validation_codes_match_the_oracle(oracle, case):
    _, V, S, start, rp, tok, nxt, acc, want = case
    a = A()
    a.V, a.S, a.start = V, S, start
    a.row_ptr, a.tok, a.next, a.accepting = (np.array(rp, np.int64), np.array(tok, np.int32),
                                             np.array(nxt, np.int32), np.array(acc, np.uint8))
    assert oracle.validate(a) == want
    rc = _compile_rc(V, S, start, rp, tok, nxt, acc)
    if want != 0:
        assert rc == want
    else:
        # valid automaton: compiles on a GPU box, fails loudly (CD_ERR_CUDA) without a device
        assert rc == (0 if torch.cuda.is_available() else 4)


def test_trie_sugar_rejects_bad_label_sets():
    for labels in ([[1, 2], [1]], [[1], [1, 2]], [[5], [5]], [[]], [[99]]):
        with pytest.raises(cd.CdError) as e:
            cd.compile_trie(16, labels)
        assert e.value.code == 2


def test_no_silent_fallback_without_a_device():
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(cd.CdError) as e:
        cd.compile_dfa(16, 2, 0, [0, 1, 1], [3], [1], [0, 1])
    assert e.value.code == 4


def test_product_package_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2606_31808_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                text = open(os.path.join(dirpath, f)).read()
                assert "oracle_cd" not in text and "import oracle" not in text and "from oracle" not in text, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            text = open(os.path.join(ROOT, "oracle", f)).read()
            assert "paper_2606_31808_b200 import" not in text and "import paper_2606_31808_b200" not in text
            assert "libcd" not in text and "cd.h" not in text
