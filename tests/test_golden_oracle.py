"""The oracle still reproduces the frozen fixtures under tests/golden/ (see
make_golden.py there for what they are and how they were written)."""
import numpy as np
import pytest

import workloads as wl
from golden_util import read_decode

CASES = {
    "c0_decode.txt": lambda: wl.CONFIGS["c0"],
    "c3_small_decode.txt": lambda: wl.scaled(wl.CONFIGS["c3"], V=4096, B=48, S=64, max_steps=10),
}


@pytest.mark.parametrize("name", sorted(CASES))
def test_oracle_matches_golden(oracle, name):
    cfg = CASES[name]()
    aut = wl.build_automaton(cfg)
    res = oracle.decode_loop(aut, wl.build_step_logits(cfg, aut))
    gold = read_decode(name)
    for k in ("tokens", "len", "done", "final_state", "n_active_hist"):
        assert np.array_equal(res[k], gold[k]), k
    np.testing.assert_allclose(res["sum_logprob"], gold["sum_logprob"], rtol=0, atol=1e-13)
