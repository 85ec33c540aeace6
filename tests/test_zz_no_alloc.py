"""cd_compact_noalloc against cd_compact (and the oracle) on the GPU.

Why the entry point exists: the library normally runs beside the LM server that produces the
logits, and that server has reserved almost all of HBM before the first query arrives.  A query
engine in that position cannot count on cudaMalloc / cudaMallocAsync while it decodes: the call may
fail for lack of memory, it may stall every stream of the device, or the memory pool it needs may
be switched off or capped.  cd_compact_noalloc runs the same multi-CTA compaction with its scratch
(one word per 4096 slots + a ticket) in a fixed 32 KB array that is part of libcd.so, so it never
allocates; the price is a limit of 2^24 slots per call and one shared array per GPU.

What is checked: integer outputs, so the bar is the one of the other compaction tests -- bit for
bit -- against cd_compact on the same inputs, and against the oracle's list filter.  Every case
calls the entry point TWICE IN A ROW with different `done` flags, because the array keeps the
previous call's chunk prefixes and tickets: a missing clear shows up in the second call, not the
first.  The file is named to be collected last (a failure here must not hide other tests under
`pytest -x`) and passes alone in a fresh process as well as after the rest of the suite: it makes
its own inputs and relies on no earlier call having touched the array.
"""
import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def cd():
    import paper_2606_31808_b200 as m

    if not torch.cuda.is_available():
        pytest.fail("no CUDA device: these tests must run on the GPU box")
    m.lib()
    return m


def _inputs(n, seed, p_done):
    rng = np.random.default_rng(seed)
    done = (rng.random(n) < p_done).astype(np.uint8)
    ids = np.sort(rng.choice(10 * n + 1, size=n, replace=False)).astype(np.int32)
    st = rng.integers(0, 5000, size=n).astype(np.int32)
    return done, ids, st


def _outputs(n):
    return (torch.full((max(n, 1),), -7, dtype=torch.int32, device="cuda:0"),
            torch.full((max(n, 1),), -7, dtype=torch.int32, device="cuda:0"),
            torch.full((1,), -7, dtype=torch.int32, device="cuda:0"))


# one chunk, a ragged second chunk, many chunks with a ragged tail; then fewer chunks than the call before
@pytest.mark.parametrize("n", [0, 1, 33, 4096, 4097, 70000, 1_000_003])
def test_two_calls_in_a_row_match_cd_compact_and_the_oracle(cd, oracle, n):
    # second call: other flags, and (for n > 4096) a shorter list, so it reuses words the first call left non-zero
    calls = [(n, 0.3, 11), (n if n <= 4096 else n - 4095, 0.8, 12)]
    for m, p_done, seed in calls:
        done, ids, st = _inputs(m, seed + m, p_done)
        d, i, s = (torch.tensor(a, device="cuda:0") for a in (done, ids, st))
        ro, so, na = cd.compact_noalloc(d, i, s, _outputs(m))
        ref_ro, ref_so, ref_na = cd.compact(d, i, s)
        k = int(ref_na)
        assert int(na) == k
        assert torch.equal(ro[:k], ref_ro[:k]) and torch.equal(so[:k], ref_so[:k])
        o_ro, o_so, o_k = oracle.compact(done, ids, st)
        assert o_k == k
        assert ro[:k].cpu().numpy().tolist() == o_ro.tolist()
        assert so[:k].cpu().numpy().tolist() == o_so.tolist()
        assert (ro[k:] == -7).all() and (so[k:] == -7).all()  # nothing written past the kept slots
        # implicit ids, no states
        ro2, _, na2 = cd.compact_noalloc(d, None, None, _outputs(m))
        assert int(na2) == k and ro2[:k].cpu().numpy().tolist() == np.flatnonzero(done == 0).tolist()


def test_the_largest_size_and_one_past_it(cd):
    n = cd.COMPACT_NOALLOC_MAX_N
    done = (torch.arange(n, device="cuda:0") % 3 == 0).to(torch.uint8)  # keeps ids with i % 3 != 0
    for _ in range(2):
        ro, _, na = cd.compact_noalloc(done, None, None, _outputs(n))
        ref_ro, _, ref_na = cd.compact(done)
        k = int(ref_na)
        assert int(na) == k == n - (n + 2) // 3
        assert torch.equal(ro[:k], ref_ro[:k])
    big = torch.zeros(n + 1, dtype=torch.uint8, device="cuda:0")
    out = _outputs(n + 1)
    with pytest.raises(cd.CdError) as e:
        cd.compact_noalloc(big, None, None, out)
    assert e.value.code == 1  # CD_ERR_ARG
    assert str(n) in str(e.value) and "cd_compact" in str(e.value)
    torch.cuda.synchronize()
    assert int(out[2]) == -7  # refused before anything was enqueued


def test_it_allocates_no_device_memory(cd):
    done, ids, st = _inputs(300_000, 5, 0.5)
    d, i, s = (torch.tensor(a, device="cuda:0") for a in (done, ids, st))
    out = _outputs(300_000)
    cd.compact_noalloc(d, i, s, out)  # set-up call of this device, if no test before this one made it
    torch.cuda.synchronize()
    # outputs are preallocated and nothing is read back inside the loop: the driver's free-memory figure must not drop
    free0, _ = torch.cuda.mem_get_info(0)
    for _ in range(50):
        cd.compact_noalloc(d, i, s, out)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info(0)
    assert free1 >= free0
    o = np.flatnonzero(done == 0)
    assert int(out[2]) == o.size and out[0][: o.size].cpu().numpy().tolist() == ids[o].tolist()
