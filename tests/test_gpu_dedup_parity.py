"""Parity of cd_dedup / cd_join_results / cd_filter_rows (through the C ABI)
with the oracle's O8 / O9: integer work, bit-exact."""
import numpy as np
import pytest
import torch

import workloads as wl

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def cd():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    import paper_2606_31808_b200 as m

    m.lib()
    return m


@pytest.mark.parametrize("N,nv,skew", [(1, 1, False), (7, 3, False), (4096, 1, False), (4097, 50, False),
                                       (20000, 2000, True), (12345, 10**9, False), (30000, 17, True)])
def test_dedup_matches_oracle(cd, oracle, N, nv, skew):
    keys = wl.make_keys(7, N, nv, skew=skew)
    rep, dr, nd = cd.dedup(keys.to("cuda:0"))
    torch.cuda.synchronize()
    o_rep, o_dr = oracle.dedup(keys.numpy())
    D = int(nd)
    assert D == o_dr.size
    assert np.array_equal(dr[:D].cpu().numpy(), o_dr)
    assert np.array_equal(rep.cpu().numpy(), o_rep)


def test_dedup_extreme_keys_and_empty(cd, oracle):
    i64 = np.iinfo(np.int64)
    keys = np.array([i64.min, 0, -1, i64.max, i64.min, -1, 7, i64.min + 1, i64.max], dtype=np.int64)
    rep, dr, nd = cd.dedup(torch.from_numpy(keys).to("cuda:0"))
    o_rep, o_dr = oracle.dedup(keys)
    assert int(nd) == o_dr.size and np.array_equal(dr[: int(nd)].cpu().numpy(), o_dr)
    assert np.array_equal(rep.cpu().numpy(), o_rep)
    rep, dr, nd = cd.dedup(torch.zeros(0, dtype=torch.int64, device="cuda:0"))
    assert int(nd) == 0


def test_dedup_full_size_properties(cd, oracle):
    """N = 2^20 rows, 4096 distinct values (N = 10^6, |dom| << N), the size bench.py
    times.  The oracle's quadratic scan does not finish here, so: properties that determine the
    result (join key reproduces every row's value; first rows ascending, map to themselves and are
    first occurrences) on every row, and the oracle itself on a prefix."""
    N, nv = 1 << 20, 4096
    keys = wl.make_keys(4, N, nv, device="cuda:0", skew=True)
    rep, dr, nd = cd.dedup(keys)
    torch.cuda.synchronize()
    D = int(nd)
    dr = dr[:D].long()
    assert torch.equal(keys[dr[rep.long()]], keys)
    assert bool((dr[1:] > dr[:-1]).all())
    assert torch.equal(rep[dr].long(), torch.arange(D, device="cuda:0"))
    assert torch.unique(keys[dr]).numel() == D == torch.unique(keys).numel()
    # first occurrence: no earlier row carries the same value  <=>  min row index per value == dr
    mins = torch.full((D,), N, dtype=torch.int64, device="cuda:0")
    mins.scatter_reduce_(0, rep.long(), torch.arange(N, device="cuda:0"), reduce="amin")
    assert torch.equal(mins, dr)
    P = 20000
    o_rep, o_dr = oracle.dedup(keys[:P].cpu().numpy())
    assert np.array_equal(rep[:P].cpu().numpy(), o_rep)  # a prefix dedups to a prefix
    assert np.array_equal(dr[: o_dr.size].cpu().numpy(), o_dr)


def test_dedup_decode_join_equals_decoding_every_row(cd, oracle):
    """The whole optimisation: dedup -> decode the distinct rows -> join back, against
    the oracle decoding every row."""
    V, nv, N, steps = 2048, 40, 700, 6
    aut = wl.make_random_dfa(33, V, 12, 0.1, 0.15)
    dfa = cd.compile_dfa(aut.V, aut.S, aut.start, aut.row_ptr, aut.tok, aut.next, aut.accepting, device="cuda:0")
    keys = wl.make_keys(33, N, nv)
    rep, dr, nd = cd.dedup(keys.to("cuda:0"))
    D = int(nd)
    per_value = [wl.make_logits(33, k, D, V, 2.0, torch.bfloat16) for k in range(steps)]
    res_d = cd.decode_loop(dfa, [x.to("cuda:0") for x in per_value])
    got = cd.join_results(rep, res_d)
    torch.cuda.synchronize()
    full = [x[rep.cpu().long()] for x in per_value]
    want = oracle.decode_loop(aut, full)
    for k in ("tokens", "len", "final_state", "done"):
        assert np.array_equal(got[k].cpu().numpy(), want[k]), k
    err = np.abs(got["sum_logprob"].cpu().numpy().astype(np.float64) - want["sum_logprob"])
    assert np.all(err <= 1e-5 * (want["len"] + np.abs(want["sum_logprob"])) + 1e-12)
    o_join = oracle.join_results(rep.cpu().numpy(), {k: v.cpu().numpy() for k, v in res_d.items()})
    for k in ("tokens", "len", "final_state", "done"):
        assert np.array_equal(got[k].cpu().numpy(), o_join[k]), k
    assert np.array_equal(got["sum_logprob"].cpu().numpy(), o_join["sum_logprob"].astype(np.float32))


@pytest.mark.parametrize("N", [1, 33, 4096, 5000, 70000])
def test_filter_rows_matches_oracle(cd, oracle, N):
    aut = wl.make_random_dfa(35, 512, 23, 0.2, 0.3)
    dfa = cd.compile_dfa(aut.V, aut.S, aut.start, aut.row_ptr, aut.tok, aut.next, aut.accepting, device="cuda:0")
    rng = np.random.default_rng(N)
    sat = ((rng.random(aut.S) < 0.5) & (np.asarray(aut.accepting) != 0)).astype(np.uint8)
    dfa.set_satisfying(sat)
    fs = rng.integers(0, aut.S, N).astype(np.int32)
    dn = (rng.random(N) < 0.8).astype(np.uint8)
    ids = rng.permutation(N).astype(np.int32)
    for row_ids in (None, ids):
        ro, no = cd.filter_rows(dfa, torch.from_numpy(fs).to("cuda:0"), torch.from_numpy(dn).to("cuda:0"),
                                None if row_ids is None else torch.from_numpy(row_ids).to("cuda:0"))
        want = oracle.filter_rows(fs, dn, sat, row_ids=row_ids)
        assert int(no) == want.size
        assert np.array_equal(ro[: int(no)].cpu().numpy(), want)


@pytest.mark.parametrize("max_steps", [1, 4, 6, 8, 16, 20, 132, 256])
@pytest.mark.parametrize("N,D", [(1, 1), (33, 5), (70001, 977)])
def test_join_copies_token_rows_of_every_width(cd, oracle, max_steps, N, D):
    """LEFT JOIN back for histories of any length: rows of whole 16-byte vectors move as int4 with a
    group of lanes per row (max_steps % 4 == 0: 1, 2, 4 ... 32 lanes), the others element by element; same result
    as the oracle's O9, bit for bit, including an unaligned view of the history (element-wise path again)."""
    rng = np.random.default_rng(max_steps * 1000 + N)
    res_d = {
        "tokens": torch.tensor(rng.integers(-1, 262144, size=(D, max_steps)).astype(np.int32), device="cuda:0"),
        "len": torch.tensor(rng.integers(0, max_steps + 1, size=D).astype(np.int32), device="cuda:0"),
        "final_state": torch.tensor(rng.integers(0, 4096, size=D).astype(np.int32), device="cuda:0"),
        "sum_logprob": torch.tensor(rng.normal(size=D).astype(np.float32), device="cuda:0"),
        "done": torch.tensor(rng.integers(0, 2, size=D).astype(np.uint8), device="cuda:0"),
    }
    rep = torch.tensor(rng.integers(0, D, size=N).astype(np.int32), device="cuda:0")
    want = oracle.join_results(rep.cpu().numpy(), {k: v.cpu().numpy() for k, v in res_d.items()})
    got = cd.join_results(rep, res_d)
    torch.cuda.synchronize()
    for k in ("tokens", "len", "final_state", "done"):
        assert np.array_equal(got[k].cpu().numpy(), want[k]), k
    assert np.array_equal(got["sum_logprob"].cpu().numpy(), want["sum_logprob"].astype(np.float32))
    # the same history at an address that is not a multiple of 16 bytes
    flat = torch.empty(D * max_steps + 1, dtype=torch.int32, device="cuda:0")
    shifted = flat[1:].view(D, max_steps)
    shifted.copy_(res_d["tokens"])
    got2 = cd.join_results(rep, dict(res_d, tokens=shifted))
    assert np.array_equal(got2["tokens"].cpu().numpy(), want["tokens"])
