"""ctypes loader for oracle_cd.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Argument marshalling only: every number the oracle reports is computed in
oracle_cd.c (plain C, single thread, double accumulation).
This module shares nothing with paper_2606_31808_b200/ and must never be
imported from it.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from typing import List, Optional, Sequence, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "oracle_cd.c")
_SO = os.path.join(_HERE, "liboracle_cd.so")
_SO_SAN = os.path.join(_HERE, "liboracle_cd_san.so")
_lib = None

F32, BF16 = 0, 1
OK, ERR_ARG, ERR_AUTOMATON, ERR_DEAD_STATE = 0, 1, 2, 3


class OracleError(RuntimeError):
    def __init__(self, code: int):
        super().__init__(f"oracle status {code}")
        self.code = code


def build(force: bool = False, sanitize: bool = False) -> str:
    """gcc -O2 the oracle into oracle/liboracle_cd.so (no -ffast-math: the
    summation order and exp/log are the definition).  sanitize=True builds
    oracle/liboracle_cd_san.so with AddressSanitizer + UndefinedBehaviorSanitizer
    (loaded by a process started with LD_PRELOAD=libasan and
    ORACLE_CD_SANITIZE=1, see tests/test_oracle_sanitized.py)."""
    so = _SO_SAN if sanitize else _SO
    if force or not os.path.exists(so) or os.path.getmtime(so) < os.path.getmtime(_SRC):
        tmp = so + f".tmp{os.getpid()}"
        flags = ["-O1", "-g", "-fsanitize=address,undefined", "-fno-omit-frame-pointer"] if sanitize else ["-O2"]
        subprocess.check_call(
            ["gcc"] + flags + ["-ffp-contract=off", "-std=c11", "-fPIC", "-shared", "-Wall", "-Wextra", "-o", tmp, _SRC, "-lm"]
        )
        os.replace(tmp, so)
    return so


def asan_runtime() -> str:
    """Path of gcc's libasan.so (to LD_PRELOAD into the python process that loads the sanitized oracle)."""
    return subprocess.check_output(["gcc", "-print-file-name=libasan.so"], text=True).strip()


def _load():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build(sanitize=os.environ.get("ORACLE_CD_SANITIZE") == "1"))
        _lib.orc_validate.restype = C.c_int
        _lib.orc_step.restype = C.c_int
        _lib.orc_compact.restype = C.c_int
        _lib.orc_decode_loop.restype = C.c_int
        _lib.orc_decode_loop_limit.restype = C.c_int
        _lib.orc_head_step.restype = C.c_int
        _lib.orc_head_decode_loop.restype = C.c_int
        _lib.orc_dedup.restype = C.c_int
        _lib.orc_sample_step.restype = C.c_int
        _lib.orc_sample_decode_loop.restype = C.c_int
        _lib.orc_det_logf.restype = C.c_float
        _lib.orc_det_logf.argtypes = [C.c_float]
        _lib.orc_fmix32.restype = C.c_uint32
        _lib.orc_fmix32.argtypes = [C.c_uint32]
        _lib.orc_gumbel.restype = C.c_float
        _lib.orc_gumbel.argtypes = [C.c_uint32] * 5
        _lib.orc_join_results.restype = C.c_int
        _lib.orc_filter_rows.restype = C.c_int
        _lib.orc_head_logit.restype = C.c_double
    return _lib


def _p(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _csr(aut):
    """aut: anything with V, S, start, row_ptr, tok, next, accepting (torch or numpy)."""
    def np_(x, dt):
        if hasattr(x, "detach"):
            x = x.detach().cpu().numpy()
        return np.ascontiguousarray(np.asarray(x, dtype=dt))
    return (
        int(aut.V), int(aut.S), int(aut.start),
        np_(aut.row_ptr, np.int64), np_(aut.tok, np.int32), np_(aut.next, np.int32),
        np_(aut.accepting, np.uint8),
    )


def _logits_np(x) -> Tuple[np.ndarray, int]:
    """[rows, ld] logits (torch fp32 / bf16 tensor, or numpy float32 / uint16
    holding bf16 bits) -> contiguous numpy array + dtype code.  Bytes are
    passed through untouched."""
    if hasattr(x, "detach"):
        import torch
        x = x.detach().cpu().contiguous()
        if x.dtype == torch.bfloat16:
            return x.view(torch.int16).numpy().view(np.uint16), BF16
        if x.dtype == torch.float32:
            return x.numpy(), F32
        raise TypeError(f"unsupported logits dtype {x.dtype}")
    x = np.ascontiguousarray(x)
    if x.dtype == np.uint16:
        return x, BF16
    if x.dtype == np.float32:
        return x, F32
    raise TypeError(f"unsupported logits dtype {x.dtype}")


def validate(aut) -> int:
    V, S, start, rp, tok, nxt, acc = _csr(aut)
    return int(_load().orc_validate(C.c_int32(V), C.c_int32(S), C.c_int32(start), _p(rp), _p(tok), _p(nxt), _p(acc)))


def step(aut, logits, state: Sequence[int], row_map: Optional[Sequence[int]] = None):
    """One constrained step (O2).  Returns (token i32[n], logprob f64[n],
    lse f64[n], done u8[n], new_state i32[n])."""
    V, S, start, rp, tok, nxt, acc = _csr(aut)
    x, dt = _logits_np(logits)
    assert x.ndim == 2
    ld = x.shape[1]
    st = np.ascontiguousarray(np.asarray(state, dtype=np.int32)).copy()
    n = st.shape[0]
    rm = None if row_map is None else np.ascontiguousarray(np.asarray(row_map, dtype=np.int32))
    if rm is not None:
        assert rm.shape[0] == n and (n == 0 or (rm.min() >= 0 and rm.max() < x.shape[0]))
    else:
        assert n <= x.shape[0]
    token = np.empty(n, np.int32)
    lp = np.empty(n, np.float64)
    lse = np.empty(n, np.float64)
    done = np.empty(n, np.uint8)
    rc = _load().orc_step(
        C.c_int32(V), C.c_int32(S), _p(rp), _p(tok), _p(nxt), _p(acc), _p(x), C.c_int(dt),
        C.c_int64(ld), _p(rm), _p(st), C.c_int32(n), _p(token), _p(lp), _p(lse), _p(done))
    if rc != OK:
        raise OracleError(rc)
    return token, lp, lse, done, st


def compact(done, row_ids=None, state=None):
    """Stable compaction (O3).  Returns (row_ids_out i32[k], state_out i32[k] or None, k)."""
    dn = np.ascontiguousarray(np.asarray(done, dtype=np.uint8))
    n = dn.shape[0]
    ri = None if row_ids is None else np.ascontiguousarray(np.asarray(row_ids, dtype=np.int32))
    si = None if state is None else np.ascontiguousarray(np.asarray(state, dtype=np.int32))
    ro = np.empty(n, np.int32)
    so = None if si is None else np.empty(n, np.int32)
    k = C.c_int32(0)
    rc = _load().orc_compact(_p(dn), _p(ri), _p(si), C.c_int32(n), _p(ro), _p(so), C.byref(k))
    if rc != OK:
        raise OracleError(rc)
    return ro[: k.value].copy(), (None if so is None else so[: k.value].copy()), int(k.value)


def decode_loop(aut, step_logits: List, max_steps: Optional[int] = None, satisfying=None, limit: int = 0,
                satisfied: int = 0):
    """The whole loop (O4).  step_logits[k] is [B, ld] indexed by original row
    id.  Returns dict(tokens i32[B,max_steps], len, final_state, sum_logprob
    f64, done u8, n_active_hist i32[max_steps]).  With `satisfying` (u8[S]) the
    LIMIT early exit of O5 applies: `satisfied` rows counted so far in, the new
    count out under key "satisfied"."""
    V, S, start, rp, tok, nxt, acc = _csr(aut)
    max_steps = len(step_logits) if max_steps is None else max_steps
    assert len(step_logits) >= max_steps
    arrs = [_logits_np(x) for x in step_logits[:max_steps]]
    if max_steps:
        B, ld = arrs[0][0].shape
        dt = arrs[0][1]
        assert all(a.shape == (B, ld) and d == dt for a, d in arrs)
    else:
        B, ld, dt = 0, V, F32
    ptrs = (C.c_void_p * max(1, max_steps))(*[a.ctypes.data for a, _ in arrs])
    tokens = np.empty((B, max_steps), np.int32)
    ln = np.empty(B, np.int32)
    fs = np.empty(B, np.int32)
    slp = np.empty(B, np.float64)
    done = np.empty(B, np.uint8)
    hist = np.zeros(max(1, max_steps), np.int32)
    sat = None if satisfying is None else np.ascontiguousarray(np.asarray(satisfying, dtype=np.uint8))
    if sat is not None:
        assert sat.shape[0] == S
    cnt = C.c_int32(int(satisfied))
    rc = _load().orc_decode_loop_limit(
        C.c_int32(V), C.c_int32(S), C.c_int32(start), _p(rp), _p(tok), _p(nxt), _p(acc), ptrs,
        C.c_int(dt), C.c_int64(ld), C.c_int32(B), C.c_int32(max_steps), _p(tokens), _p(ln), _p(fs),
        _p(slp), _p(done), _p(hist), _p(sat), C.c_int32(int(limit)), C.byref(cnt) if sat is not None else None)
    if rc != OK:
        raise OracleError(rc)
    return dict(tokens=tokens, len=ln, final_state=fs, sum_logprob=slp, done=done,
                n_active_hist=hist[:max_steps], satisfied=int(cnt.value))


def _bf16_np(x) -> np.ndarray:
    """[rows, ld] bf16 (torch tensor, or numpy uint16 holding the bits) -> contiguous uint16 array."""
    if hasattr(x, "detach"):
        import torch
        x = x.detach().cpu().contiguous()
        assert x.dtype == torch.bfloat16
        return x.view(torch.int16).numpy().view(np.uint16)
    x = np.ascontiguousarray(x)
    assert x.dtype == np.uint16
    return x


def head_step(aut, hidden, W, H: int, state: Sequence[int], row_map: Optional[Sequence[int]] = None):
    """One constrained step on x = hidden @ W[:, :H].T (O6).  hidden [rows, ldh] and
    W [V, ldw] are bf16.  Returns (token, logprob f64, lse f64, done, new_state, gap f64)."""
    V, S, start, rp, tok, nxt, acc = _csr(aut)
    hd = _bf16_np(hidden)
    w = _bf16_np(W)
    assert hd.ndim == 2 and w.ndim == 2 and w.shape[0] == V
    st = np.ascontiguousarray(np.asarray(state, dtype=np.int32)).copy()
    n = st.shape[0]
    rm = None if row_map is None else np.ascontiguousarray(np.asarray(row_map, dtype=np.int32))
    if rm is not None:
        assert rm.shape[0] == n and (n == 0 or (rm.min() >= 0 and rm.max() < hd.shape[0]))
    else:
        assert n <= hd.shape[0]
    token = np.empty(n, np.int32)
    lp = np.empty(n, np.float64)
    lse = np.empty(n, np.float64)
    done = np.empty(n, np.uint8)
    gap = np.empty(n, np.float64)
    rc = _load().orc_head_step(
        C.c_int32(V), C.c_int32(S), _p(rp), _p(tok), _p(nxt), _p(acc), _p(hd), C.c_int64(hd.shape[1]),
        _p(w), C.c_int64(w.shape[1]), C.c_int32(H), _p(rm), _p(st), C.c_int32(n), _p(token), _p(lp),
        _p(lse), _p(done), _p(gap))
    if rc != OK:
        raise OracleError(rc)
    return token, lp, lse, done, st, gap


def head_logit(hidden, W, H: int, row: int, token: int) -> float:
    """<hidden[row, :H], W[token, :H]> in double (O6)."""
    hd = _bf16_np(hidden)
    w = _bf16_np(W)
    hrow = np.ascontiguousarray(hd[row])
    return float(_load().orc_head_logit(_p(hrow), _p(w), C.c_int64(w.shape[1]), C.c_int32(H), C.c_int32(token)))


def head_decode_loop(aut, step_hidden: List, W, H: int, max_steps: Optional[int] = None):
    """The loop on the LM-head step (O7).  step_hidden[k] is [B, ldh] bf16 indexed by original row id."""
    V, S, start, rp, tok, nxt, acc = _csr(aut)
    max_steps = len(step_hidden) if max_steps is None else max_steps
    assert 1 <= max_steps <= len(step_hidden)
    arrs = [_bf16_np(x) for x in step_hidden[:max_steps]]
    w = _bf16_np(W)
    B, ldh = arrs[0].shape
    assert all(a.shape == (B, ldh) for a in arrs) and w.shape[0] == V
    ptrs = (C.c_void_p * max_steps)(*[a.ctypes.data for a in arrs])
    tokens = np.empty((B, max_steps), np.int32)
    ln = np.empty(B, np.int32)
    fs = np.empty(B, np.int32)
    slp = np.empty(B, np.float64)
    done = np.empty(B, np.uint8)
    hist = np.zeros(max_steps, np.int32)
    rc = _load().orc_head_decode_loop(
        C.c_int32(V), C.c_int32(S), C.c_int32(start), _p(rp), _p(tok), _p(nxt), _p(acc), ptrs, C.c_int64(ldh),
        _p(w), C.c_int64(w.shape[1]), C.c_int32(H), C.c_int32(B), C.c_int32(max_steps), _p(tokens), _p(ln), _p(fs),
        _p(slp), _p(done), _p(hist))
    if rc != OK:
        raise OracleError(rc)
    return dict(tokens=tokens, len=ln, final_state=fs, sum_logprob=slp, done=done, n_active_hist=hist)


def dedup(keys):
    """SELECT DISTINCT in first-occurrence order (O8).  Returns (rep i32[N], distinct_rows i32[D])."""
    k = np.ascontiguousarray(np.asarray(keys, dtype=np.int64))
    N = k.shape[0]
    rep = np.empty(N, np.int32)
    dr = np.empty(max(N, 1), np.int32)
    D = C.c_int32(0)
    rc = _load().orc_dedup(_p(k), C.c_int32(N), _p(rep), _p(dr), C.byref(D))
    if rc != OK:
        raise OracleError(rc)
    return rep, dr[: D.value].copy()


def join_results(rep, res: dict):
    """LEFT JOIN of the distinct values' decode results back to the rows (O8)."""
    r = np.ascontiguousarray(np.asarray(rep, dtype=np.int32))
    N = r.shape[0]
    tk = np.ascontiguousarray(res["tokens"], dtype=np.int32)
    ms = tk.shape[1]
    ln = np.ascontiguousarray(res["len"], dtype=np.int32)
    fs = np.ascontiguousarray(res["final_state"], dtype=np.int32)
    slp = np.ascontiguousarray(res["sum_logprob"], dtype=np.float64)
    dn = np.ascontiguousarray(res["done"], dtype=np.uint8)
    out = dict(tokens=np.empty((N, ms), np.int32), len=np.empty(N, np.int32), final_state=np.empty(N, np.int32),
               sum_logprob=np.empty(N, np.float64), done=np.empty(N, np.uint8))
    rc = _load().orc_join_results(_p(r), C.c_int32(N), C.c_int32(ms), _p(tk), _p(ln), _p(fs), _p(slp), _p(dn),
                                  _p(out["tokens"]), _p(out["len"]), _p(out["final_state"]), _p(out["sum_logprob"]),
                                  _p(out["done"]))
    if rc != OK:
        raise OracleError(rc)
    return out


def filter_rows(final_state, done, satisfying, row_ids=None):
    """Cascade filter (O9): ids of the rows that finished in a satisfying state, order kept."""
    fs = np.ascontiguousarray(np.asarray(final_state, dtype=np.int32))
    dn = np.ascontiguousarray(np.asarray(done, dtype=np.uint8))
    sat = np.ascontiguousarray(np.asarray(satisfying, dtype=np.uint8))
    ri = None if row_ids is None else np.ascontiguousarray(np.asarray(row_ids, dtype=np.int32))
    N = fs.shape[0]
    out = np.empty(max(N, 1), np.int32)
    k = C.c_int32(0)
    rc = _load().orc_filter_rows(_p(fs), _p(dn), _p(ri), C.c_int32(N), _p(sat), C.c_int32(sat.shape[0]), _p(out), C.byref(k))
    if rc != OK:
        raise OracleError(rc)
    return out[: k.value].copy()


def det_logf(x: float) -> float:
    """The fp32 logarithm of the sampling definition (O10)."""
    return float(_load().orc_det_logf(C.c_float(x)))


def fmix32(h: int) -> int:
    """The 32-bit mixing function of the counter-based generator (O10)."""
    return int(_load().orc_fmix32(h & 0xFFFFFFFF))


def gumbel(seed: int, row: int, step: int, tok: int) -> float:
    """Gumbel noise of (seed, row, step, token) (O10)."""
    return float(_load().orc_gumbel(seed & 0xFFFFFFFF, (seed >> 32) & 0xFFFFFFFF, row, step, tok))


def sample_step(aut, logits, state: Sequence[int], temperature: float, seed: int, step: int = 0,
                row_map: Optional[Sequence[int]] = None):
    """One sampled step (O10).  Returns (token, logprob f64, lse f64, done, new_state)."""
    V, S, start, rp, tok, nxt, acc = _csr(aut)
    x, dt = _logits_np(logits)
    ld = x.shape[1]
    st = np.ascontiguousarray(np.asarray(state, dtype=np.int32)).copy()
    n = st.shape[0]
    rm = None if row_map is None else np.ascontiguousarray(np.asarray(row_map, dtype=np.int32))
    token = np.empty(n, np.int32)
    lp = np.empty(n, np.float64)
    lse = np.empty(n, np.float64)
    done = np.empty(n, np.uint8)
    rc = _load().orc_sample_step(
        C.c_int32(V), C.c_int32(S), _p(rp), _p(tok), _p(nxt), _p(acc), _p(x), C.c_int(dt), C.c_int64(ld), _p(rm),
        _p(st), C.c_int32(n), C.c_float(temperature), C.c_uint64(seed), C.c_int32(step), _p(token), _p(lp), _p(lse),
        _p(done))
    if rc != OK:
        raise OracleError(rc)
    return token, lp, lse, done, st


def sample_decode_loop(aut, step_logits: List, temperature: float, seed: int, step_base: int = 0,
                       max_steps: Optional[int] = None):
    """The loop with sampled steps (O4 on O10)."""
    V, S, start, rp, tok, nxt, acc = _csr(aut)
    max_steps = len(step_logits) if max_steps is None else max_steps
    arrs = [_logits_np(x) for x in step_logits[:max_steps]]
    B, ld = arrs[0][0].shape
    dt = arrs[0][1]
    ptrs = (C.c_void_p * max_steps)(*[a.ctypes.data for a, _ in arrs])
    tokens = np.empty((B, max_steps), np.int32)
    ln = np.empty(B, np.int32)
    fs = np.empty(B, np.int32)
    slp = np.empty(B, np.float64)
    done = np.empty(B, np.uint8)
    rc = _load().orc_sample_decode_loop(
        C.c_int32(V), C.c_int32(S), C.c_int32(start), _p(rp), _p(tok), _p(nxt), _p(acc), ptrs, C.c_int(dt),
        C.c_int64(ld), C.c_int32(B), C.c_int32(max_steps), C.c_float(temperature), C.c_uint64(seed),
        C.c_int32(step_base), _p(tokens), _p(ln), _p(fs), _p(slp), _p(done))
    if rc != OK:
        raise OracleError(rc)
    return dict(tokens=tokens, len=ln, final_state=fs, sum_logprob=slp, done=done)
