"""ctypes binding with the same names as include/cd.h (argument marshalling only)."""
from __future__ import annotations

import ctypes as C
import os
from typing import List, Optional, Sequence

import torch

HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(HERE, "libcd.so")
_lib = None

F32, BF16 = 0, 1
LOOP_AUTO, LOOP_PER_STEP, LOOP_BARRIER = 0, 1, 2
STATUS = {0: "CD_OK", 1: "CD_ERR_ARG", 2: "CD_ERR_AUTOMATON", 3: "CD_ERR_DEAD_STATE",
          4: "CD_ERR_CUDA", 5: "CD_ERR_OOM", 6: "CD_ERR_INTERNAL"}

# every symbol include/cd.h declares (tests check the .so exports each of them)
SYMBOLS = (
    "cd_compile_dfa", "cd_build_trie", "cd_compile_trie", "cd_build_list", "cd_set_loop_mode", "cd_loop_trace", "cd_compile_list", "cd_free_dfa", "cd_dfa_info", "cd_set_gather_max", "cd_set_sampling", "cd_reserve", "cd_step",
    "cd_transition", "cd_compact", "cd_compact_noalloc", "cd_decode_loop", "cd_decode_loop_async", "cd_loop_sync", "cd_set_satisfying", "cd_set_limit", "cd_decode_loop_limit", "cd_decode_loop_host", "cd_set_head_gather_max", "cd_head_step", "cd_head_decode_loop", "cd_head_decode_loop_host", "cd_probe_read", "cd_decode_loop_cb", "cd_head_decode_loop_cb", "cd_dedup", "cd_join_results", "cd_filter_rows", "cd_launch_count",
    "cd_last_error",
)


class CdError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"{STATUS.get(code, code)}: {msg}")
        self.code = code


def lib_path() -> str:
    return _SO


def lib():
    """Loads libcd.so; fails loudly when it has not been built (no fallback)."""
    global _lib
    if _lib is None:
        if not os.path.exists(_SO):
            raise RuntimeError(
                f"{_SO} is missing: build it with `python -m paper_2606_31808_b200.build` "
                "(nvcc, sm_100a). There is no CPU fallback.")
        L = C.CDLL(_SO)
        for name in SYMBOLS:
            getattr(L, name)
        L.cd_last_error.restype = C.c_char_p
        L.cd_launch_count.restype = C.c_int64
        L.cd_free_dfa.restype = None
        L.cd_free_dfa.argtypes = [C.c_void_p]
        for name in SYMBOLS:
            if name not in ("cd_last_error", "cd_launch_count", "cd_free_dfa"):
                getattr(L, name).restype = C.c_int
        _lib = L
    return _lib


def _check(rc: int):
    if rc != 0:
        raise CdError(rc, lib().cd_last_error().decode("utf-8", "replace"))


def launch_count() -> int:
    return int(lib().cd_launch_count())


def _host(x, dtype) -> torch.Tensor:
    t = torch.as_tensor(x).detach().to("cpu", dtype).contiguous()
    return t


def _ptr(t: Optional[torch.Tensor]):
    return C.c_void_p(None) if t is None else C.c_void_p(t.data_ptr())


def _stream(device) -> C.c_void_p:
    return C.c_void_p(torch.cuda.current_stream(device).cuda_stream)


def _dt(t: torch.Tensor) -> int:
    if t.dtype == torch.bfloat16:
        return BF16
    if t.dtype == torch.float32:
        return F32
    raise TypeError(f"logits must be float32 or bfloat16, got {t.dtype}")


def _dev_tensor(t: torch.Tensor, dtype, name: str, device) -> torch.Tensor:
    if t.dtype != dtype or not t.is_cuda or not t.is_contiguous() or t.device != device:
        raise TypeError(f"{name}: expected contiguous {dtype} tensor on {device}")
    return t


class Dfa:
    """Owner of a cd_dfa_t* handle."""

    def __init__(self, handle: int, device: torch.device):
        self._h = C.c_void_p(handle)
        self.device = device
        V, S, start = C.c_int32(), C.c_int32(), C.c_int32()
        nnz, mb = C.c_int64(), C.c_int64()
        _check(lib().cd_dfa_info(self._h, C.byref(V), C.byref(S), C.byref(start), C.byref(nnz), C.byref(mb)))
        self.V, self.S, self.start, self.nnz, self.mask_bytes = V.value, S.value, start.value, nnz.value, mb.value

    def set_gather_max(self, max_transitions: int):
        """cd_set_gather_max: 0 = dense scan only, > 0 threshold, -1 automatic."""
        _check(lib().cd_set_gather_max(self._h, C.c_int32(max_transitions)))

    def set_sampling(self, temperature: float, seed: int = 0, step_base: int = 0):
        """cd_set_sampling: temperature 0 = greedy; > 0 = seeded Gumbel-max sampling."""
        _check(lib().cd_set_sampling(self._h, C.c_float(temperature), C.c_uint64(seed), C.c_int32(step_base)))

    def set_head_gather_max(self, max_transitions: int):
        """cd_set_head_gather_max: 0 = dense contraction for every state, > 0 threshold, -1 automatic."""
        _check(lib().cd_set_head_gather_max(self._h, C.c_int32(max_transitions)))

    def set_loop_mode(self, mode: int):
        """cd_set_loop_mode: LOOP_AUTO (one persistent kernel per decode loop when possible: row groups that advance
        independently, or the lock-step kernel when a LIMIT is set), LOOP_BARRIER (the lock-step persistent kernel)
        or LOOP_PER_STEP (one launch per decoding step)."""
        _check(lib().cd_set_loop_mode(self._h, C.c_int32(mode)))

    def loop_trace(self, cap: int = 256):
        """cd_loop_trace: (active rows, nanoseconds) per decoding step of the last persistent loop on the
        current stream, as two python lists (empty if that loop ran as per-step launches)."""
        t = (C.c_int64 * max(cap, 1))()
        n = (C.c_int32 * max(cap, 1))()
        steps = C.c_int32(0)
        _check(lib().cd_loop_trace(self._h, _stream(self.device), C.c_int32(cap), t, n, C.byref(steps)))
        k = min(steps.value, cap)
        return [int(n[i]) for i in range(k)], [int(t[i]) for i in range(k)]

    def set_satisfying(self, satisfying):
        """cd_set_satisfying: u8[S] host flags (None clears)."""
        if satisfying is None:
            _check(lib().cd_set_satisfying(self._h, C.c_void_p(None)))
            return
        t = _host(satisfying, torch.uint8)
        if t.numel() != self.S:
            raise ValueError("satisfying must have S entries")
        _check(lib().cd_set_satisfying(self._h, _ptr(t)))

    def set_limit(self, limit: int, satisfied: Optional[torch.Tensor]):
        """cd_set_limit: LIMIT early exit for every loop; satisfied = device int32[1] counter (None clears)."""
        if satisfied is not None:
            _dev_tensor(satisfied, torch.int32, "satisfied", self.device)
        self._limit_ctr = satisfied  # keep the counter alive
        _check(lib().cd_set_limit(self._h, C.c_int32(limit), _ptr(satisfied)))

    def reserve(self, max_rows: int):
        _check(lib().cd_reserve(self._h, C.c_int32(max_rows), _stream(self.device)))

    def close(self):
        if self._h:
            lib().cd_free_dfa(self._h)
            self._h = C.c_void_p(None)

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def _device_index(device) -> torch.device:
    d = torch.device(device)
    if d.type != "cuda":
        raise ValueError("device must be a CUDA device")
    return torch.device("cuda", d.index if d.index is not None else torch.cuda.current_device())


def compile_dfa(V: int, S: int, start: int, row_ptr, tok, next, accepting, device="cuda") -> Dfa:
    """cd_compile_dfa: host CSR in, device automaton store out."""
    L = lib()
    rp, tk = _host(row_ptr, torch.int64), _host(tok, torch.int32)
    nx, ac = _host(next, torch.int32), _host(accepting, torch.uint8)
    if rp.numel() != S + 1 or ac.numel() != S or tk.numel() != nx.numel():
        raise ValueError("CSR array lengths do not match S / nnz")
    if S >= 0 and rp.numel() > 0 and int(rp[-1]) > tk.numel():
        raise ValueError("row_ptr[S] exceeds len(tok)")
    dev_index = 0
    dev = None
    if torch.cuda.is_available():
        dev = _device_index(device)
        dev_index = dev.index
    out = C.c_void_p()
    _check(L.cd_compile_dfa(C.c_int32(V), C.c_int32(S), C.c_int32(start), _ptr(rp), _ptr(tk), _ptr(nx),
                            _ptr(ac), C.c_int(dev_index), C.byref(out)))
    return Dfa(out.value, dev)


def _label_args(labels):
    ptr = [0]
    flat: List[int] = []
    for lab in labels:
        flat.extend(int(t) for t in lab)
        ptr.append(len(flat))
    return torch.tensor(ptr, dtype=torch.int64), torch.tensor(flat if flat else [0], dtype=torch.int32)


def build_trie(V: int, labels: Sequence[Sequence[int]], eos: int = -1):
    """cd_build_trie (host only, no device needed): the CSR of the option-set automaton as
    (S, row_ptr i64[S+1], tok i32[nnz], next i32[nnz], accepting u8[S]); eos >= 0 = the EOS / longest-match variant."""
    lp, lt = _label_args(labels)
    head = [C.c_int32(V), C.c_int32(len(labels)), _ptr(lp), _ptr(lt), C.c_int32(eos)]
    S, nnz = C.c_int32(0), C.c_int64(0)
    null = C.c_void_p(None)
    _check(lib().cd_build_trie(*head, C.byref(S), C.byref(nnz), null, null, null, null))
    rp = torch.empty(S.value + 1, dtype=torch.int64)
    tk = torch.empty(max(nnz.value, 1), dtype=torch.int32)
    nx = torch.empty(max(nnz.value, 1), dtype=torch.int32)
    ac = torch.empty(S.value, dtype=torch.uint8)
    _check(lib().cd_build_trie(*head, C.byref(S), C.byref(nnz), _ptr(rp), _ptr(tk), _ptr(nx), _ptr(ac)))
    return S.value, rp, tk[: nnz.value], nx[: nnz.value], ac


def compile_trie(V: int, labels: Sequence[Sequence[int]], device="cuda", eos: int = -1) -> Dfa:
    """cd_compile_trie: option-set / boolean types as a trie over token-id labels (eos >= 0: labels may be
    prefixes of one another, every row ends with eos in the one accepting sink)."""
    L = lib()
    lp, lt = _label_args(labels)
    dev_index = 0
    dev = None
    if torch.cuda.is_available():
        dev = _device_index(device)
        dev_index = dev.index
    out = C.c_void_p()
    _check(L.cd_compile_trie(C.c_int32(V), C.c_int32(len(labels)), _ptr(lp), _ptr(lt), C.c_int32(eos), C.c_int(dev_index),
                             C.byref(out)))
    return Dfa(out.value, dev)


def step(dfa: Dfa, logits: torch.Tensor, state: torch.Tensor, row_map: Optional[torch.Tensor] = None,
         n: Optional[int] = None, want_lse: bool = True, out=None):
    """cd_step on torch's current stream.  state (int32, device) is updated in
    place.  Returns (token i32[n], logprob f32[n], lse f32[n] or None, done u8[n]);
    `out` may pass those four buffers in (each with at least n elements)."""
    dev = dfa.device
    if logits.dim() != 2 or not logits.is_cuda or logits.stride(1) != 1:
        raise TypeError("logits must be a 2-D CUDA tensor with unit inner stride")
    _dev_tensor(state, torch.int32, "state", dev)
    n = state.numel() if n is None else n
    if row_map is not None:
        _dev_tensor(row_map, torch.int32, "row_map", dev)
    if out is not None:
        token, logprob, lse, done = out
    else:
        token = torch.empty(n, dtype=torch.int32, device=dev)
        logprob = torch.empty(n, dtype=torch.float32, device=dev)
        lse = torch.empty(n, dtype=torch.float32, device=dev) if want_lse else None
        done = torch.empty(n, dtype=torch.uint8, device=dev)
    _check(lib().cd_step(dfa._h, _ptr(logits), C.c_int(_dt(logits)), C.c_int64(logits.stride(0)), _ptr(row_map),
                         _ptr(state), C.c_int32(n), _ptr(token), _ptr(logprob), _ptr(lse), _ptr(done),
                         _stream(dev)))
    return token, logprob, lse, done


def head_step(dfa: Dfa, hidden: torch.Tensor, W: torch.Tensor, state: torch.Tensor,
              row_map: Optional[torch.Tensor] = None, n: Optional[int] = None, H: Optional[int] = None,
              want_lse: bool = True, out=None):
    """cd_head_step on torch's current stream: the constrained step on x = hidden[:, :H] @ W[:, :H].T
    without materialising x.  hidden [rows, ldh] and W [V, ldw] are bf16 CUDA tensors with unit inner
    stride; state (int32, device) is updated in place.  Returns (token, logprob, lse or None, done)."""
    dev = dfa.device
    for name, t in (("hidden", hidden), ("W", W)):
        if t.dim() != 2 or not t.is_cuda or t.stride(1) != 1 or t.dtype != torch.bfloat16:
            raise TypeError(f"{name} must be a 2-D bf16 CUDA tensor with unit inner stride")
    H = hidden.shape[1] if H is None else H
    if W.shape[0] != dfa.V or W.shape[1] < H or hidden.shape[1] < H:
        raise ValueError("W must be [V, >= H] and hidden [rows, >= H]")
    _dev_tensor(state, torch.int32, "state", dev)
    n = state.numel() if n is None else n
    if row_map is not None:
        _dev_tensor(row_map, torch.int32, "row_map", dev)
    if out is not None:
        token, logprob, lse, done = out
    else:
        token = torch.empty(n, dtype=torch.int32, device=dev)
        logprob = torch.empty(n, dtype=torch.float32, device=dev)
        lse = torch.empty(n, dtype=torch.float32, device=dev) if want_lse else None
        done = torch.empty(n, dtype=torch.uint8, device=dev)
    _check(lib().cd_head_step(dfa._h, _ptr(hidden), C.c_int64(hidden.stride(0)), _ptr(W), C.c_int64(W.stride(0)),
                              C.c_int32(H), _ptr(row_map), _ptr(state), C.c_int32(n), _ptr(token), _ptr(logprob),
                              _ptr(lse), _ptr(done), _stream(dev)))
    return token, logprob, lse, done


def transition(dfa: Dfa, token: torch.Tensor, state: torch.Tensor):
    """cd_transition: state updated in place; returns done u8[n]."""
    dev = dfa.device
    _dev_tensor(token, torch.int32, "token", dev)
    _dev_tensor(state, torch.int32, "state", dev)
    n = state.numel()
    done = torch.empty(n, dtype=torch.uint8, device=dev)
    _check(lib().cd_transition(dfa._h, _ptr(token), _ptr(state), C.c_int32(n), _ptr(done), _stream(dev)))
    return done


def compact(done: torch.Tensor, row_ids: Optional[torch.Tensor] = None, state: Optional[torch.Tensor] = None,
            n: Optional[int] = None, out=None):
    """cd_compact.  Returns (row_ids_out i32[n], state_out i32[n] or None,
    n_active device int32[1]); only the first n_active entries are meaningful."""
    dev = done.device
    _dev_tensor(done, torch.uint8, "done", dev)
    n = done.numel() if n is None else n
    if row_ids is not None:
        _dev_tensor(row_ids, torch.int32, "row_ids", dev)
    if state is not None:
        _dev_tensor(state, torch.int32, "state", dev)
    if out is not None:
        ro, so, na = out
    else:
        ro = torch.empty(max(n, 1), dtype=torch.int32, device=dev)
        so = torch.empty(max(n, 1), dtype=torch.int32, device=dev) if state is not None else None
        na = torch.empty(1, dtype=torch.int32, device=dev)
    with torch.cuda.device(dev):
        _check(lib().cd_compact(_ptr(done), _ptr(row_ids), _ptr(state), C.c_int32(n), _ptr(ro), _ptr(so), _ptr(na),
                                _stream(dev)))
    return ro, so, na


COMPACT_NOALLOC_MAX_N = 1 << 24


def compact_noalloc(done: torch.Tensor, row_ids: Optional[torch.Tensor], state: Optional[torch.Tensor], out,
                    n: Optional[int] = None):
    """cd_compact_noalloc: `compact` for processes that may not allocate device memory while they
    decode -- an engine living beside an LM server that has reserved almost all of HBM, or one
    whose stream-ordered memory pool is disabled or capped.  The scan's scratch is a fixed 32 KB
    array inside libcd.so, so the library allocates nothing; for the same reason this wrapper
    allocates nothing either: `out` = (row_ids_out i32[>= n], state_out i32[>= n] or None,
    n_active i32[1]) is required and returned.  At most COMPACT_NOALLOC_MAX_N slots per call
    (CdError with code CD_ERR_ARG above that).  All calls on a GPU share the array: keep them
    on one stream.  Make the first call on each GPU during set-up, before any stream capture."""
    dev = done.device
    _dev_tensor(done, torch.uint8, "done", dev)
    n = done.numel() if n is None else n
    if row_ids is not None:
        _dev_tensor(row_ids, torch.int32, "row_ids", dev)
    if state is not None:
        _dev_tensor(state, torch.int32, "state", dev)
    ro, so, na = out
    with torch.cuda.device(dev):
        _check(lib().cd_compact_noalloc(_ptr(done), _ptr(row_ids), _ptr(state), C.c_int32(n), _ptr(ro), _ptr(so),
                                        _ptr(na), _stream(dev)))
    return ro, so, na


def _loop_outputs(B: int, max_steps: int, device, pin: bool = False):
    kw = dict(device=device)
    if pin:
        kw = dict(device="cpu", pin_memory=True)
    return dict(
        tokens=torch.empty((B, max_steps), dtype=torch.int32, **kw),
        len=torch.empty(B, dtype=torch.int32, **kw),
        final_state=torch.empty(B, dtype=torch.int32, **kw),
        sum_logprob=torch.empty(B, dtype=torch.float32, **kw),
        done=torch.empty(B, dtype=torch.uint8, **kw),
    )


def decode_loop(dfa: Dfa, step_logits: Sequence[torch.Tensor], max_steps: Optional[int] = None, out=None,
                limit: Optional[int] = None, satisfied: Optional[torch.Tensor] = None):
    """cd_decode_loop: step_logits[k] are [B, ld] CUDA tensors indexed by original
    row id.  Returns dict(tokens, len, final_state, sum_logprob, done) of device
    tensors.  Synchronises the current stream once.  With `limit` and the device
    int32[1] counter `satisfied` it is cd_decode_loop_limit."""
    dev = dfa.device
    max_steps = len(step_logits) if max_steps is None else max_steps
    if max_steps > len(step_logits):
        raise ValueError("fewer step buffers than max_steps")
    if max_steps == 0:
        raise ValueError("max_steps must be >= 1 here (B is taken from the step buffers)")
    x0 = step_logits[0]
    B, ld, dt = x0.shape[0], x0.stride(0), _dt(x0)
    for x in step_logits[:max_steps]:
        if x.dim() != 2 or not x.is_cuda or x.stride(1) != 1 or x.shape[0] != B or x.stride(0) != ld or _dt(x) != dt:
            raise TypeError("step_logits must share shape, stride and dtype")
    ptrs = (C.c_void_p * max_steps)(*[x.data_ptr() for x in step_logits[:max_steps]])
    out = _loop_outputs(B, max_steps, dev) if out is None else out
    if limit is not None:
        _dev_tensor(satisfied, torch.int32, "satisfied", dev)
        _check(lib().cd_decode_loop_limit(dfa._h, ptrs, C.c_int(dt), C.c_int64(ld), C.c_int32(B), C.c_int32(max_steps),
                                          _ptr(out["tokens"]), _ptr(out["len"]), _ptr(out["final_state"]),
                                          _ptr(out["sum_logprob"]), _ptr(out["done"]), C.c_int32(limit),
                                          _ptr(satisfied), _stream(dev)))
        return out
    _check(lib().cd_decode_loop(dfa._h, ptrs, C.c_int(dt), C.c_int64(ld), C.c_int32(B), C.c_int32(max_steps),
                                _ptr(out["tokens"]), _ptr(out["len"]), _ptr(out["final_state"]),
                                _ptr(out["sum_logprob"]), _ptr(out["done"]), _stream(dev)))
    return out


class PreparedLoop:
    """The arguments of a cd_decode_loop call marshalled once: run() / enqueue() only make the C call (a decode
    loop over a small batch lasts tens of microseconds, less than building its ctypes arguments).  The step
    buffers, the outputs and the stream (torch's current one at construction) are fixed."""

    def __init__(self, dfa: Dfa, step_logits: Sequence[torch.Tensor], max_steps: Optional[int] = None, out=None):
        dev = dfa.device
        max_steps = len(step_logits) if max_steps is None else max_steps
        if max_steps > len(step_logits) or max_steps == 0:
            raise ValueError("need 1 <= max_steps <= len(step_logits)")
        x0 = step_logits[0]
        B, ld, dt = x0.shape[0], x0.stride(0), _dt(x0)
        for x in step_logits[:max_steps]:
            if x.dim() != 2 or not x.is_cuda or x.stride(1) != 1 or x.shape[0] != B or x.stride(0) != ld or _dt(x) != dt:
                raise TypeError("step_logits must share shape, stride and dtype")
        self.dfa = dfa
        self._keep = list(step_logits[:max_steps])
        self._ptrs = (C.c_void_p * max_steps)(*[x.data_ptr() for x in self._keep])
        self.out = _loop_outputs(B, max_steps, dev) if out is None else out
        self._stream = _stream(dev)
        self._args = (dfa._h, self._ptrs, C.c_int(dt), C.c_int64(ld), C.c_int32(B), C.c_int32(max_steps),
                      _ptr(self.out["tokens"]), _ptr(self.out["len"]), _ptr(self.out["final_state"]),
                      _ptr(self.out["sum_logprob"]), _ptr(self.out["done"]), self._stream)
        self._run = lib().cd_decode_loop
        self._enqueue = lib().cd_decode_loop_async

    def run(self):
        """cd_decode_loop (synchronises the stream once)."""
        _check(self._run(*self._args))
        return self.out

    def enqueue(self):
        """cd_decode_loop_async: enqueue only; the outputs are valid after sync()."""
        _check(self._enqueue(*self._args))
        return self.out

    def sync(self):
        """cd_loop_sync: synchronise the stream and report the device-side status of the loops enqueued on it."""
        _check(lib().cd_loop_sync(self.dfa._h, self._stream))
        return self.out


def decode_loop_async(dfa: Dfa, step_logits: Sequence[torch.Tensor], max_steps: Optional[int] = None, out=None):
    """cd_decode_loop_async: as decode_loop but only enqueued on torch's current stream; call loop_sync(dfa)
    before reading the outputs."""
    return PreparedLoop(dfa, step_logits, max_steps, out).enqueue()


def loop_sync(dfa: Dfa):
    """cd_loop_sync on torch's current stream."""
    _check(lib().cd_loop_sync(dfa._h, _stream(dfa.device)))


def head_decode_loop_host(dfa: Dfa, step_hidden_host: Sequence[torch.Tensor], W: torch.Tensor,
                          H: Optional[int] = None, max_steps: Optional[int] = None, out=None):
    """cd_head_decode_loop_host: HOST hidden states in (pinned memory overlaps the copies), device W,
    HOST outputs; the host<->device copies happen inside the call."""
    dev = dfa.device
    max_steps = len(step_hidden_host) if max_steps is None else max_steps
    h0 = step_hidden_host[0]
    B, ldh = h0.shape[0], h0.stride(0)
    H = h0.shape[1] if H is None else H
    for h in step_hidden_host[:max_steps]:
        if h.is_cuda or h.dim() != 2 or h.stride(1) != 1 or h.dtype != torch.bfloat16 or h.shape[0] != B or h.stride(0) != ldh:
            raise TypeError("step_hidden_host must be host bf16 tensors sharing shape and stride")
    if not W.is_cuda or W.dtype != torch.bfloat16 or W.stride(1) != 1 or W.shape[0] != dfa.V:
        raise TypeError("W must be a [V, ld] bf16 CUDA tensor")
    ptrs = (C.c_void_p * max_steps)(*[h.data_ptr() for h in step_hidden_host[:max_steps]])
    out = _loop_outputs(B, max_steps, dev, pin=True) if out is None else out
    _check(lib().cd_head_decode_loop_host(dfa._h, ptrs, C.c_int64(ldh), _ptr(W), C.c_int64(W.stride(0)), C.c_int32(H),
                                          C.c_int32(B), C.c_int32(max_steps), _ptr(out["tokens"]), _ptr(out["len"]),
                                          _ptr(out["final_state"]), _ptr(out["sum_logprob"]), _ptr(out["done"]),
                                          _stream(dev)))
    return out


def head_decode_loop(dfa: Dfa, step_hidden: Sequence[torch.Tensor], W: torch.Tensor, H: Optional[int] = None,
                     max_steps: Optional[int] = None, out=None):
    """cd_head_decode_loop: step_hidden[k] are [B, ldh] bf16 CUDA tensors (hidden states of step k,
    indexed by original row id), W [V, ldw] bf16.  Returns dict(tokens, len, final_state, sum_logprob,
    done) of device tensors."""
    dev = dfa.device
    max_steps = len(step_hidden) if max_steps is None else max_steps
    if max_steps == 0 or max_steps > len(step_hidden):
        raise ValueError("need 1 <= max_steps <= len(step_hidden)")
    h0 = step_hidden[0]
    B, ldh = h0.shape[0], h0.stride(0)
    H = h0.shape[1] if H is None else H
    for h in list(step_hidden[:max_steps]) + [W]:
        if h.dim() != 2 or not h.is_cuda or h.stride(1) != 1 or h.dtype != torch.bfloat16:
            raise TypeError("hidden states and W must be 2-D bf16 CUDA tensors with unit inner stride")
    for h in step_hidden[:max_steps]:
        if h.shape[0] != B or h.stride(0) != ldh:
            raise TypeError("step_hidden must share shape and stride")
    if W.shape[0] != dfa.V:
        raise ValueError("W must have V rows")
    ptrs = (C.c_void_p * max_steps)(*[h.data_ptr() for h in step_hidden[:max_steps]])
    out = _loop_outputs(B, max_steps, dev) if out is None else out
    _check(lib().cd_head_decode_loop(dfa._h, ptrs, C.c_int64(ldh), _ptr(W), C.c_int64(W.stride(0)), C.c_int32(H),
                                     C.c_int32(B), C.c_int32(max_steps), _ptr(out["tokens"]), _ptr(out["len"]),
                                     _ptr(out["final_state"]), _ptr(out["sum_logprob"]), _ptr(out["done"]),
                                     _stream(dev)))
    return out


def decode_loop_host(dfa: Dfa, step_logits_host: Sequence[torch.Tensor], max_steps: Optional[int] = None, out=None):
    """cd_decode_loop_host: HOST tensors in (pinned memory overlaps the copies),
    HOST tensors out; host<->device copies happen inside the call."""
    dev = dfa.device
    max_steps = len(step_logits_host) if max_steps is None else max_steps
    x0 = step_logits_host[0]
    B, ld, dt = x0.shape[0], x0.stride(0), _dt(x0)
    for x in step_logits_host[:max_steps]:
        if x.is_cuda or x.dim() != 2 or x.stride(1) != 1 or x.shape[0] != B or x.stride(0) != ld or _dt(x) != dt:
            raise TypeError("step_logits_host must be host tensors sharing shape, stride and dtype")
    ptrs = (C.c_void_p * max_steps)(*[x.data_ptr() for x in step_logits_host[:max_steps]])
    out = _loop_outputs(B, max_steps, dev, pin=True) if out is None else out
    _check(lib().cd_decode_loop_host(dfa._h, ptrs, C.c_int(dt), C.c_int64(ld), C.c_int32(B), C.c_int32(max_steps),
                                     _ptr(out["tokens"]), _ptr(out["len"]), _ptr(out["final_state"]),
                                     _ptr(out["sum_logprob"]), _ptr(out["done"]), _stream(dev)))
    return out


def dedup(keys: torch.Tensor, out=None):
    """cd_dedup: keys int64[N] on the device -> (rep i32[N], distinct_rows i32[N], n_distinct i32[1]);
    only the first n_distinct entries of distinct_rows are meaningful."""
    if keys.dtype != torch.int64 or not keys.is_cuda or not keys.is_contiguous() or keys.dim() != 1:
        raise TypeError("keys must be a contiguous 1-D int64 CUDA tensor")
    dev = keys.device
    N = keys.numel()
    if out is not None:
        rep, dr, nd = out
    else:
        rep = torch.empty(max(N, 1), dtype=torch.int32, device=dev)
        dr = torch.empty(max(N, 1), dtype=torch.int32, device=dev)
        nd = torch.empty(1, dtype=torch.int32, device=dev)
    with torch.cuda.device(dev):
        _check(lib().cd_dedup(_ptr(keys), C.c_int32(N), _ptr(rep), _ptr(dr), _ptr(nd), _stream(dev)))
    return rep[:N], dr, nd


def join_results(rep: torch.Tensor, res: dict, out=None):
    """cd_join_results: broadcast the distinct values' loop outputs (dict of device tensors) to the rows."""
    dev = rep.device
    _dev_tensor(rep, torch.int32, "rep", dev)
    N = rep.numel()
    ms = res["tokens"].shape[1]
    out = _loop_outputs(N, ms, dev) if out is None else out
    with torch.cuda.device(dev):
        _check(lib().cd_join_results(_ptr(rep), C.c_int32(N), C.c_int32(ms), _ptr(res["tokens"]), _ptr(res["len"]),
                                     _ptr(res["final_state"]), _ptr(res["sum_logprob"]), _ptr(res["done"]),
                                     _ptr(out["tokens"]), _ptr(out["len"]), _ptr(out["final_state"]),
                                     _ptr(out["sum_logprob"]), _ptr(out["done"]), _stream(dev)))
    return out


def filter_rows(dfa: Dfa, final_state: torch.Tensor, done: torch.Tensor, row_ids: Optional[torch.Tensor] = None):
    """cd_filter_rows: (row_ids_out i32[N], n_out i32[1]) of the rows that finished in a satisfying state."""
    dev = dfa.device
    _dev_tensor(final_state, torch.int32, "final_state", dev)
    _dev_tensor(done, torch.uint8, "done", dev)
    if row_ids is not None:
        _dev_tensor(row_ids, torch.int32, "row_ids", dev)
    N = final_state.numel()
    ro = torch.empty(max(N, 1), dtype=torch.int32, device=dev)
    no = torch.empty(1, dtype=torch.int32, device=dev)
    _check(lib().cd_filter_rows(dfa._h, _ptr(final_state), _ptr(done), _ptr(row_ids), C.c_int32(N), _ptr(ro), _ptr(no),
                                _stream(dev)))
    return ro, no


def probe_read(buf: torch.Tensor, iters: int = 10) -> float:
    """cd_probe_read: GB/s of a pure-read pass over `buf` with the step kernel's copy machinery."""
    if not buf.is_cuda or not buf.is_contiguous():
        raise TypeError("buf must be a contiguous CUDA tensor")
    nbytes = buf.numel() * buf.element_size()
    ms = C.c_float(0.0)
    with torch.cuda.device(buf.device):
        _check(lib().cd_probe_read(_ptr(buf), C.c_int64(nbytes), C.c_int32(iters), C.byref(ms), _stream(buf.device)))
    return (nbytes // 8192 * 8192) / (ms.value * 1e-3) / 1e9


_NEXT_FN = C.CFUNCTYPE(C.c_int, C.c_void_p, C.c_int32, C.c_void_p, C.c_void_p, C.c_int32, C.POINTER(C.c_void_p),
                       C.POINTER(C.c_int64), C.POINTER(C.c_int32))


def _wrap_next(fn, dev, B, keep):
    """fn(step, row_ids i32[B] device view, n_active i32[1] device view) -> (tensor [rows, ld], by_slot)."""
    def thunk(user, step, d_ids, d_n, n_upper, out_ptr, out_ld, out_by_slot):
        try:
            ids = _view_i32(d_ids, n_upper, dev)
            n = _view_i32(d_n, 1, dev)
            t, by_slot = fn(int(step), ids, n)
            if t.dim() != 2 or not t.is_cuda or t.stride(1) != 1:
                return 2
            keep.append(t)  # the buffer must outlive the loop
            out_ptr[0] = t.data_ptr()
            out_ld[0] = t.stride(0)
            out_by_slot[0] = 1 if by_slot else 0
            return 0
        except Exception:  # never raise through the C ABI
            import traceback
            traceback.print_exc()
            return 1
    return _NEXT_FN(thunk)


def _view_i32(ptr: int, n: int, dev) -> torch.Tensor:
    """Zero-copy int32 view of device memory owned by the library (valid during the callback's loop)."""
    class _Holder:
        pass
    h = _Holder()
    h.__cuda_array_interface__ = {"shape": (n,), "typestr": "<i4", "data": (int(ptr), False), "version": 3}
    return torch.as_tensor(h, device=dev)


def decode_loop_cb(dfa: Dfa, next_logits, dtype: torch.dtype, B: int, max_steps: int, out=None):
    """cd_decode_loop_cb: next_logits(step, row_ids, n_active) -> (logits tensor, by_slot) is called before
    every step and must only enqueue work on torch's current stream."""
    dev = dfa.device
    keep: List[torch.Tensor] = []
    cb = _wrap_next(next_logits, dev, B, keep)
    out = _loop_outputs(B, max_steps, dev) if out is None else out
    dt = BF16 if dtype == torch.bfloat16 else F32
    _check(lib().cd_decode_loop_cb(dfa._h, cb, C.c_void_p(None), C.c_int(dt), C.c_int32(B), C.c_int32(max_steps),
                                   _ptr(out["tokens"]), _ptr(out["len"]), _ptr(out["final_state"]),
                                   _ptr(out["sum_logprob"]), _ptr(out["done"]), _stream(dev)))
    return out


def head_decode_loop_cb(dfa: Dfa, next_hidden, W: torch.Tensor, H: int, B: int, max_steps: int, out=None):
    """cd_head_decode_loop_cb: next_hidden(step, row_ids, n_active) -> (hidden bf16 tensor, by_slot)."""
    dev = dfa.device
    keep: List[torch.Tensor] = []
    cb = _wrap_next(next_hidden, dev, B, keep)
    out = _loop_outputs(B, max_steps, dev) if out is None else out
    _check(lib().cd_head_decode_loop_cb(dfa._h, cb, C.c_void_p(None), _ptr(W), C.c_int64(W.stride(0)), C.c_int32(H),
                                        C.c_int32(B), C.c_int32(max_steps), _ptr(out["tokens"]), _ptr(out["len"]),
                                        _ptr(out["final_state"]), _ptr(out["sum_logprob"]), _ptr(out["done"]),
                                        _stream(dev)))
    return out


def _list_args(V, labels, open_, sep, close, min_items, max_items, eos=-1):
    ptr, flat = [0], []
    for lab in labels:
        flat.extend(int(t) for t in lab)
        ptr.append(len(flat))
    lp = torch.tensor(ptr, dtype=torch.int64)
    lt = torch.tensor(flat if flat else [0], dtype=torch.int32)
    ts = [torch.tensor(list(x) if len(x) else [0], dtype=torch.int32) for x in (open_, sep, close)]
    args = [C.c_int32(V), C.c_int32(len(labels)), _ptr(lp), _ptr(lt), _ptr(ts[0]), C.c_int32(len(open_)), _ptr(ts[1]),
            C.c_int32(len(sep)), _ptr(ts[2]), C.c_int32(len(close)), C.c_int32(min_items), C.c_int32(max_items),
            C.c_int32(eos)]
    return args, (lp, lt, ts)


def build_list(V: int, labels: Sequence[Sequence[int]], open_: Sequence[int], sep: Sequence[int],
               close: Sequence[int], min_items: int, max_items: int, eos: int = -1):
    """cd_build_list (host only, no device needed): the CSR of the quantified-list automaton as
    (S, row_ptr i64[S+1], tok i32[nnz], next i32[nnz], accepting u8[S])."""
    args, keep = _list_args(V, labels, open_, sep, close, min_items, max_items, eos)
    S, nnz = C.c_int32(0), C.c_int64(0)
    null = C.c_void_p(None)
    _check(lib().cd_build_list(*args, C.byref(S), C.byref(nnz), null, null, null, null))
    rp = torch.empty(S.value + 1, dtype=torch.int64)
    tk = torch.empty(max(nnz.value, 1), dtype=torch.int32)
    nx = torch.empty(max(nnz.value, 1), dtype=torch.int32)
    ac = torch.empty(S.value, dtype=torch.uint8)
    _check(lib().cd_build_list(*args, C.byref(S), C.byref(nnz), _ptr(rp), _ptr(tk), _ptr(nx), _ptr(ac)))
    return S.value, rp, tk[: nnz.value], nx[: nnz.value], ac


def compile_list(V: int, labels: Sequence[Sequence[int]], open_: Sequence[int], sep: Sequence[int],
                 close: Sequence[int], min_items: int, max_items: int, device="cuda", eos: int = -1) -> Dfa:
    """cd_compile_list: collection type with a quantifier ({min_items, max_items} items of an option set)."""
    args, keep = _list_args(V, labels, open_, sep, close, min_items, max_items, eos)
    dev_index, dev = 0, None
    if torch.cuda.is_available():
        dev = _device_index(device)
        dev_index = dev.index
    out = C.c_void_p()
    _check(lib().cd_compile_list(*args, C.c_int(dev_index), C.byref(out)))
    return Dfa(out.value, dev)
