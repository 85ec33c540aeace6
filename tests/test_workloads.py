"""Host-side checks of the seeded input generators (workloads/): determinism,
scalar/tensor hash agreement, CSR well-formedness, the recipe's statistics."""
import math

import numpy as np
import torch

import workloads as wl


def test_hash_scalar_and_tensor_agree():
    a = torch.arange(0, 50, dtype=torch.int64)
    b = torch.arange(1000, 1050, dtype=torch.int64)
    for seed, salt in [(0, 0), (3, 1), (123456, 77)]:
        ht = wl.mix32_t(seed, salt, a, b).tolist()
        hi = [wl.mix32_i(seed, salt, int(x), int(y)) for x, y in zip(a.tolist(), b.tolist())]
        assert ht == hi
        assert all(0 <= h < 2**32 for h in hi)


def test_random_dfa_is_valid_deterministic_and_has_the_stated_density(oracle):
    a = wl.make_random_dfa(seed=3, V=8192, S=96, density=0.02, accept_frac=0.10)
    b = wl.make_random_dfa(seed=3, V=8192, S=96, density=0.02, accept_frac=0.10, states_per_chunk=7)
    for f in ("row_ptr", "tok", "next", "accepting"):
        assert torch.equal(getattr(a, f), getattr(b, f))  # chunking does not change the bits
    assert oracle.validate(a) == 0
    assert a.accepting[0] == 0
    per_state = (a.row_ptr[1:] - a.row_ptr[:-1]).float()
    mean = 8192 * 0.02
    assert abs(float(per_state.mean()) - mean) < 4 * math.sqrt(mean / 96) + 1
    acc = float(a.accepting.float().mean())
    assert 0.02 < acc < 0.25
    c = wl.make_random_dfa(seed=4, V=8192, S=96, density=0.02, accept_frac=0.10)
    assert not torch.equal(a.tok[:100], c.tok[:100])


def test_sparse_dfa_never_leaves_a_dead_state(oracle):
    a = wl.make_random_dfa(seed=9, V=64, S=200, density=0.01, accept_frac=0.05)
    assert oracle.validate(a) == 0
    deg = a.row_ptr[1:] - a.row_ptr[:-1]
    assert bool(((deg > 0) | (a.accepting == 1)).all())


def test_labels_prefix_free_and_trie_shape():
    labs = wl.draw_labels(seed=2, V=50, K=20, min_len=1, max_len=3)  # tiny V forces re-draws
    assert len(labs) == 20
    for i, x in enumerate(labs):
        for j, y in enumerate(labs):
            if i != j:
                n = min(len(x), len(y))
                assert x[:n] != y[:n]
    t = wl.make_trie(50, labs)
    assert int(t.accepting.sum()) == 20
    assert t.S == 1 + len({tuple(l[:k]) for l in labs for k in range(1, len(l) + 1)})
    assert t.nnz == t.S - 1


def test_logits_recipe():
    x = wl.make_logits(1, 0, 64, 4096, 2.0, torch.bfloat16, bias_tokens=[5, 9], bias=4.0)
    y = wl.make_logits(1, 0, 64, 4096, 2.0, torch.bfloat16, bias_tokens=[5, 9], bias=4.0)
    assert torch.equal(x.view(torch.int16), y.view(torch.int16))
    z = wl.make_logits(1, 1, 64, 4096, 2.0, torch.bfloat16)
    assert not torch.equal(x.view(torch.int16), z.view(torch.int16))
    xf = x.float()
    assert abs(float(xf[:, 100:].std()) - 2.0) < 0.05
    assert abs(float(xf[:, 5].mean()) - 4.0) < 1.2
    p = wl.make_logits(1, 0, 8, 100, 1.0, torch.float32, ld=128)
    assert p.shape == (8, 128) and float(p[:, 100:].abs().max()) == 0.0


def test_configs_match_baseline_json():
    c = wl.CONFIGS
    assert (c["c0"].B, c["c0"].V, c["c0"].max_steps, c["c0"].labels) == (4, 1024, 8, [[17, 3], [42]])
    assert (c["c1"].B, c["c1"].V, c["c1"].max_steps, c["c1"].K) == (256, 262144, 4, 2)
    assert (c["c2"].B, c["c2"].V, c["c2"].K, c["c2"].max_len) == (1024, 262144, 50, 6)
    assert (c["c3"].B, c["c3"].S, c["c3"].density, c["c3"].accept_frac, c["c3"].max_steps) == (512, 512, 0.02, 0.10, 32)
    assert (c["c4"].B, c["c4"].S, c["c4"].density, c["c4"].accept_frac, c["c4"].max_steps, c["c4"].n_batches) == (
        4096, 4096, 0.005, 0.05, 16, 256)
    assert c["c4"].B * c["c4"].n_batches == 1048576


def test_shard_rows_partition():
    for B in (0, 1, 7, 4096, 4097):
        for w in (1, 2, 3, 8):
            spans = [wl.shard_rows(B, w, r) for r in range(w)]
            assert spans[0][0] == 0 and spans[-1][1] == B
            assert all(spans[i][1] == spans[i + 1][0] for i in range(w - 1))
            sizes = [b - a for a, b in spans]
            assert max(sizes) - min(sizes) <= 1
