"""Seeded synthetic inputs for the constrained-decoding hot path.

This module serves BOTH the CPU oracle (``oracle/``) and the CUDA path
(``paper_2606_31808_b200/``) and therefore holds NONE of the method's
arithmetic: no masking, no softmax, no argmax, no transition lookup, no
compaction.  It only produces

  * token-level automata in host CSR form (tries for boolean / enum typed LM
    functions, random DFAs for regex-shaped types), and
  * logits tensors,

for the five workloads of BASELINE.json ``configs[0..4]`` (SURVEY.md section
8(d) table; the paper's workloads they stand in for are the boolean ``LLMMap``
filters, k-way ``options`` classifiers and regex-shaped return types of
PAPER.md section 2.3, and section 4.2).  The paper's own data,
tokenizer and weights are not available, so every input is synthetic and
seeded; the recipe is restated in DESIGN.md.

Automata come from an integer-only mixing function (``mix32``) evaluated with
torch int64 ops, so the same bits result on CPU and on CUDA tensors.  Logits
come from a seeded ``torch.Generator`` on the device they are requested on
(CPU and CUDA generators differ: generate once, copy the bytes to the other
side, never regenerate).
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Dict, List, Optional, Sequence, Tuple

import torch

M32 = 0xFFFFFFFF
_C1 = 0x85EBCA6B
_C2 = 0xC2B2AE35
_K_SEED = 0x9E3779B1
_K_SALT = 0x27D4EB2F
_K_TOK = 0xC2B2AE3D


# --------------------------------------------------------------------------
# integer-only hash (python ints and torch int64 tensors give the same bits)
# --------------------------------------------------------------------------
def _mul32_t(h: torch.Tensor, c: int) -> torch.Tensor:
    """(h * c) mod 2^32 for 0 <= h < 2^32 held in int64, without int64 overflow."""
    lo = (h & 0xFFFF) * c
    hi = (((h >> 16) * c) & 0xFFFF) << 16
    return (lo + hi) & M32


def fmix32_t(h: torch.Tensor) -> torch.Tensor:
    h = h ^ (h >> 16)
    h = _mul32_t(h, _C1)
    h = h ^ (h >> 13)
    h = _mul32_t(h, _C2)
    h = h ^ (h >> 16)
    return h


def fmix32_i(h: int) -> int:
    h &= M32
    h ^= h >> 16
    h = (h * _C1) & M32
    h ^= h >> 13
    h = (h * _C2) & M32
    h ^= h >> 16
    return h


def mix32_i(seed: int, salt: int, a: int, b: int) -> int:
    """Scalar form of the generator hash: hash of (seed, salt, a, b)."""
    h1 = fmix32_i((seed * _K_SEED + salt * _K_SALT + a) & M32)
    return fmix32_i(h1 ^ ((b * _K_TOK) & M32))


def mix32_t(seed: int, salt: int, a: torch.Tensor, b: torch.Tensor) -> torch.Tensor:
    """Tensor form (int64 in, int64 in [0, 2^32) out); broadcasts a against b."""
    base = (seed * _K_SEED + salt * _K_SALT) & M32
    h1 = fmix32_t((a + base) & M32)
    return fmix32_t(h1 ^ ((b * _K_TOK) & M32))


# --------------------------------------------------------------------------
# automata
# --------------------------------------------------------------------------
@dataclass
class Automaton:
    """Host CSR image of a token-level DFA (the argument list of cd_compile_dfa)."""

    V: int
    S: int
    start: int
    row_ptr: torch.Tensor  # int64 [S+1], cpu
    tok: torch.Tensor  # int32 [nnz], cpu, strictly increasing inside a state
    next: torch.Tensor  # int32 [nnz], cpu
    accepting: torch.Tensor  # uint8 [S], cpu
    labels: Optional[List[List[int]]] = None  # trie only: the accepted strings
    leaf_of_label: Optional[List[int]] = None  # trie only: accepting state per label
    meta: Dict[str, object] = field(default_factory=dict)

    @property
    def nnz(self) -> int:
        return int(self.tok.numel())


def make_trie(V: int, labels: Sequence[Sequence[int]]) -> Automaton:
    """Trie over token-id labels; one accepting leaf per label, states numbered
    in insertion order (root 0).  Labels must be prefix-free and distinct
    (SURVEY 8(c) G5): with shortest-accept semantics a label extending another
    label would be unreachable."""
    children: List[Dict[int, int]] = [{}]
    is_leaf = [False]
    leaf_of_label = []
    for lab in labels:
        if len(lab) == 0:
            raise ValueError("empty label")
        node = 0
        for j, t in enumerate(lab):
            if not (0 <= t < V):
                raise ValueError("token id out of range")
            if is_leaf[node]:
                raise ValueError("label set is not prefix-free")
            nxt = children[node].get(t)
            if nxt is None:
                nxt = len(children)
                children.append({})
                is_leaf.append(False)
                children[node][t] = nxt
            node = nxt
        if children[node] or is_leaf[node]:
            raise ValueError("label set is not prefix-free / has duplicates")
        is_leaf[node] = True
        leaf_of_label.append(node)
    S = len(children)
    row_ptr = [0]
    tok: List[int] = []
    nxt_l: List[int] = []
    for s in range(S):
        for t in sorted(children[s]):
            tok.append(t)
            nxt_l.append(children[s][t])
        row_ptr.append(len(tok))
    return Automaton(
        V=V,
        S=S,
        start=0,
        row_ptr=torch.tensor(row_ptr, dtype=torch.int64),
        tok=torch.tensor(tok, dtype=torch.int32),
        next=torch.tensor(nxt_l, dtype=torch.int32),
        accepting=torch.tensor([1 if x else 0 for x in is_leaf], dtype=torch.uint8),
        labels=[list(l) for l in labels],
        leaf_of_label=leaf_of_label,
    )


def draw_labels(seed: int, V: int, K: int, min_len: int, max_len: int) -> List[List[int]]:
    """K distinct, prefix-free labels of min_len..max_len token ids drawn
    uniformly from [0, V) by the integer hash; a colliding draw is re-drawn
    with the next attempt counter."""
    labels: List[List[int]] = []
    for k in range(K):
        attempt = 0
        while True:
            span = max_len - min_len + 1
            length = min_len + mix32_i(seed, 11 + attempt, k, 0) % span
            lab = [mix32_i(seed, 11 + attempt, k, 1 + j) % V for j in range(length)]
            ok = True
            for other in labels:
                n = min(len(other), len(lab))
                if other[:n] == lab[:n]:
                    ok = False
                    break
            if ok:
                labels.append(lab)
                break
            attempt += 1
            if attempt > 1000:
                raise RuntimeError("cannot draw a prefix-free label set")
    return labels


def make_random_dfa(
    seed: int,
    V: int,
    S: int,
    density: float,
    accept_frac: float,
    device: str = "cpu",
    states_per_chunk: int = 64,
) -> Automaton:
    """Random token-level DFA (BASELINE.json configs[3], configs[4]; SURVEY
    8(c) G12): token t is allowed in state s iff hash(seed, s, t) < density*2^32
    (independent Bernoulli per pair); next state = hash' mod S; state s accepts
    iff hash''(seed, s) < accept_frac*2^32, state 0 forced non-accepting.  A
    non-accepting state that comes out empty is re-hashed with the next salt."""
    thr = int(density * 4294967296.0)
    athr = int(accept_frac * 4294967296.0)
    dev = torch.device(device)
    sid = torch.arange(S, dtype=torch.int64, device=dev)
    acc = mix32_t(seed, 3, sid, torch.zeros_like(sid)) < athr
    acc[0] = False
    tid = torch.arange(V, dtype=torch.int64, device=dev)
    counts = torch.zeros(S, dtype=torch.int64)
    toks: List[torch.Tensor] = []
    nexts: List[torch.Tensor] = []
    for s0 in range(0, S, states_per_chunk):
        s1 = min(S, s0 + states_per_chunk)
        ss = sid[s0:s1]
        allowed = mix32_t(seed, 1, ss[:, None], tid[None, :]) < thr
        # re-hash empty non-accepting states (dead states are not valid automata)
        salt = 100
        while True:
            empty = (~allowed.any(dim=1)) & (~acc[s0:s1])
            if not bool(empty.any()):
                break
            idx = torch.nonzero(empty).flatten()
            allowed[idx] = mix32_t(seed, salt, ss[idx][:, None], tid[None, :]) < thr
            salt += 1
            if salt > 200:
                raise RuntimeError("density too low: cannot fill every non-accepting state")
        nz = torch.nonzero(allowed)  # row-major: sorted by (state, token)
        s_of = nz[:, 0] + s0
        t_of = nz[:, 1]
        nxt = mix32_t(seed, 2, s_of, t_of) % S
        counts[s0:s1] = allowed.sum(dim=1).cpu()
        toks.append(t_of.to(torch.int32).cpu())
        nexts.append(nxt.to(torch.int32).cpu())
        del allowed, nz, s_of, t_of, nxt
    row_ptr = torch.zeros(S + 1, dtype=torch.int64)
    row_ptr[1:] = torch.cumsum(counts, 0)
    return Automaton(
        V=V,
        S=S,
        start=0,
        row_ptr=row_ptr,
        tok=torch.cat(toks) if toks else torch.zeros(0, dtype=torch.int32),
        next=torch.cat(nexts) if nexts else torch.zeros(0, dtype=torch.int32),
        accepting=acc.to(torch.uint8).cpu(),
        meta={"density": density, "accept_frac": accept_frac, "seed": seed},
    )


# --------------------------------------------------------------------------
# logits
# --------------------------------------------------------------------------
def make_logits(
    seed: int,
    step: int,
    B: int,
    V: int,
    std: float,
    dtype: torch.dtype,
    device: str = "cpu",
    bias_tokens: Optional[Sequence[int]] = None,
    bias: float = 0.0,
    batch: int = 0,
    ld: Optional[int] = None,
    rows_per_chunk: int = 512,
    rows: Optional[Tuple[int, int]] = None,
) -> torch.Tensor:
    """One step's logits [B, ld] (ld >= V, default V): round_to_dtype(N(0, std)
    [+ bias on bias_tokens, added before rounding]).  'N(0,2)' in BASELINE.json
    is read as standard deviation 2.  The generator is
    re-seeded per (seed, batch, step) so any step can be produced on its own.
    rows = (lo, hi): only rows [lo, hi) of the batch are kept ([hi - lo, ld]); every
    chunk is still drawn, so the kept rows are byte-identical to those of the whole
    batch (a rank's shard of a batch)."""
    ld = V if ld is None else ld
    assert ld >= V
    lo, hi = (0, B) if rows is None else rows
    assert 0 <= lo <= hi <= B
    dev = torch.device(device)
    g = torch.Generator(device=dev)
    g.manual_seed((seed * 1000003 + batch * 4099 + step) & 0x7FFFFFFFFFFFFFFF)
    out = torch.empty((hi - lo, ld), dtype=dtype, device=dev)
    if ld > V:
        out[:, V:] = 0
    bt = None
    if bias_tokens is not None and len(bias_tokens) > 0:
        bt = torch.tensor(sorted(set(int(t) for t in bias_tokens)), dtype=torch.int64, device=dev)
    for r0 in range(0, B, rows_per_chunk):
        r1 = min(B, r0 + rows_per_chunk)
        if r0 >= hi:
            break
        x = torch.randn((r1 - r0, V), generator=g, dtype=torch.float32, device=dev)
        a, b = max(r0, lo), min(r1, hi)
        if a < b:
            x = x[a - r0:b - r0]
            x.mul_(std)
            if bt is not None:
                x[:, bt] += bias
            out[a - lo:b - lo, :V] = x.to(dtype)
        del x
    return out


# --------------------------------------------------------------------------
# the five workloads (BASELINE.json configs[0..4])
# --------------------------------------------------------------------------
@dataclass
class Config:
    name: str
    desc: str
    V: int
    B: int
    max_steps: int
    dtype: torch.dtype
    std: float
    seed: int
    kind: str  # "trie" | "dfa"
    n_batches: int = 1
    # trie
    labels: Optional[List[List[int]]] = None
    K: int = 0
    min_len: int = 1
    max_len: int = 1
    bias: float = 0.0
    # dfa
    S: int = 0
    density: float = 0.0
    accept_frac: float = 0.0


CONFIGS: Dict[str, Config] = {
    "c0": Config(
        name="c0",
        desc="tiny boolean: B=4, V=1024, fp32 N(0,1), trie {true:[17,3], false:[42]}, 8 steps",
        V=1024, B=4, max_steps=8, dtype=torch.float32, std=1.0, seed=0, kind="trie",
        labels=[[17, 3], [42]],
    ),
    "c1": Config(
        name="c1",
        desc="boolean filter, full vocab: B=256, V=262144, bf16 N(0,2) +4 on label starts, 2 labels of 1-2 tokens, 4 steps",
        V=262144, B=256, max_steps=4, dtype=torch.bfloat16, std=2.0, seed=1, kind="trie",
        K=2, min_len=1, max_len=2, bias=4.0,
    ),
    "c2": Config(
        name="c2",
        desc="enum classification: B=1024, V=262144, bf16 N(0,2), trie over K=50 labels of 1-6 tokens, decode to accept",
        V=262144, B=1024, max_steps=6, dtype=torch.bfloat16, std=2.0, seed=2, kind="trie",
        K=50, min_len=1, max_len=6,
    ),
    "c3": Config(
        name="c3",
        desc="regex-shaped: B=512, V=262144, bf16 N(0,3), random DFA S=512, 2% allowed, 10% accepting, 32 steps",
        V=262144, B=512, max_steps=32, dtype=torch.bfloat16, std=3.0, seed=3, kind="dfa",
        S=512, density=0.02, accept_frac=0.10,
    ),
    "c4": Config(
        name="c4",
        desc="large table: 1,048,576 rows as 256 batches of B=4096, V=262144, bf16 N(0,2), random DFA S=4096, 0.5% allowed, 5% accepting, 16 steps",
        V=262144, B=4096, max_steps=16, dtype=torch.bfloat16, std=2.0, seed=4, kind="dfa",
        S=4096, density=0.005, accept_frac=0.05, n_batches=256,
    ),
}


def scaled(cfg: Config, **kw) -> Config:
    """A copy of cfg with some fields replaced (tests run reduced V/B/S variants
    of the same recipe so the oracle finishes in seconds)."""
    d = dict(cfg.__dict__)
    d.update(kw)
    return Config(**d)


def build_automaton(cfg: Config, device: str = "cpu") -> Automaton:
    if cfg.kind == "trie":
        labels = cfg.labels
        if labels is None:
            labels = draw_labels(cfg.seed, cfg.V, cfg.K, cfg.min_len, cfg.max_len)
        return make_trie(cfg.V, labels)
    return make_random_dfa(cfg.seed, cfg.V, cfg.S, cfg.density, cfg.accept_frac, device=device)


def bias_tokens_of(cfg: Config, aut: Automaton) -> List[int]:
    if cfg.bias == 0.0 or aut.labels is None:
        return []
    return [lab[0] for lab in aut.labels]


def build_step_logits(
    cfg: Config, aut: Automaton, device: str = "cpu", batch: int = 0,
    steps: Optional[int] = None, B: Optional[int] = None, rows: Optional[Tuple[int, int]] = None,
) -> List[torch.Tensor]:
    """The list step_logits[k] ([B, V], indexed by ORIGINAL row id) of one batch (rows = (lo, hi): that
    shard of it, see make_logits)."""
    steps = cfg.max_steps if steps is None else steps
    B = cfg.B if B is None else B
    bt = bias_tokens_of(cfg, aut)
    return [
        make_logits(cfg.seed, k, B, cfg.V, cfg.std, cfg.dtype, device=device,
                    bias_tokens=bt, bias=cfg.bias, batch=batch, rows=rows)
        for k in range(steps)
    ]


def shard_rows(B: int, world_size: int, rank: int) -> Tuple[int, int]:
    """Contiguous row partition [lo, hi) of rank: concatenating
    the ranks' locally compacted active lists in rank order is the global
    stable order, so the path needs no collective."""
    base, rem = divmod(B, world_size)
    lo = rank * base + min(rank, rem)
    hi = lo + base + (1 if rank < rem else 0)
    return lo, hi


# --------------------------------------------------------------------------
# LM-head inputs: final hidden states and the output embedding
# --------------------------------------------------------------------------
def make_hidden(seed: int, step: int, B: int, H: int, device: str = "cpu", batch: int = 0,
                exact: bool = False, ld: Optional[int] = None) -> torch.Tensor:
    """Final hidden states [B, ld] bf16 (ld >= H, default H) of one decoding step.
    exact=False: round_bf16(N(0,1)).  exact=True: multiples of 1/8 in [-1, 1]
    from the integer hash, so that every partial sum of a dot product with a
    make_head(exact=True) row is exactly representable in fp32 (the products are
    multiples of 1/64 and |sum| < 2^17 for H <= 2^17): the logits then do not
    depend on the order of accumulation."""
    ld = H if ld is None else ld
    assert ld >= H
    dev = torch.device(device)
    out = torch.zeros((B, ld), dtype=torch.bfloat16, device=dev)
    if exact:
        r = torch.arange(B, dtype=torch.int64, device=dev).unsqueeze(1)
        h = torch.arange(H, dtype=torch.int64, device=dev).unsqueeze(0)
        u = mix32_t(seed * 7919 + batch * 4099 + step, 11, r, h) % 17  # 0..16
        out[:, :H] = ((u.to(torch.float32) - 8.0) / 8.0).to(torch.bfloat16)
    else:
        g = torch.Generator(device=dev)
        g.manual_seed((seed * 1000003 + batch * 4099 + step + 0x5EED) & 0x7FFFFFFFFFFFFFFF)
        out[:, :H] = torch.randn((B, H), generator=g, dtype=torch.float32, device=dev).to(torch.bfloat16)
    return out


def make_head(seed: int, V: int, H: int, std: float, device: str = "cpu", exact: bool = False,
              ld: Optional[int] = None, rows_per_chunk: int = 16384) -> torch.Tensor:
    """Output embedding W [V, ld] bf16 (row t = embedding of token t; ld >= H).
    exact=False: round_bf16(N(0, std / sqrt(H))), so that logits of N(0,1) hidden
    states are ~N(0, std) like the logits of BASELINE.json configs.
    exact=True: multiples of 1/8 in [-1, 1] from the integer hash (see make_hidden)."""
    ld = H if ld is None else ld
    assert ld >= H
    dev = torch.device(device)
    out = torch.zeros((V, ld), dtype=torch.bfloat16, device=dev)
    g = torch.Generator(device=dev)
    g.manual_seed((seed * 1000003 + 0xEAD) & 0x7FFFFFFFFFFFFFFF)
    h = torch.arange(H, dtype=torch.int64, device=dev).unsqueeze(0)
    for t0 in range(0, V, rows_per_chunk):
        t1 = min(V, t0 + rows_per_chunk)
        if exact:
            t = torch.arange(t0, t1, dtype=torch.int64, device=dev).unsqueeze(1)
            u = mix32_t(seed, 12, t, h) % 17
            out[t0:t1, :H] = ((u.to(torch.float32) - 8.0) / 8.0).to(torch.bfloat16)
        else:
            x = torch.randn((t1 - t0, H), generator=g, dtype=torch.float32, device=dev)
            out[t0:t1, :H] = (x * (std / (H ** 0.5))).to(torch.bfloat16)
    return out


# --------------------------------------------------------------------------
# row keys for early deduplication
# --------------------------------------------------------------------------
def make_keys(seed: int, N: int, n_values: int, device: str = "cpu", skew: bool = False) -> torch.Tensor:
    """int64 [N] value keys of a table column with at most n_values distinct values (duplication
    factor rho ~ N / n_values: N = 10^6 rows, |dom| << N).  Row i carries value
    v_i = hash(seed, i) mod n_values (skew=True: the hash is squared down so that low value ids are
    frequent, a long-tailed column); the key is a 64-bit scramble of v_i, so keys are spread over
    the whole int64 range like hashes of strings."""
    dev = torch.device(device)
    i = torch.arange(N, dtype=torch.int64, device=dev)
    z = torch.zeros_like(i)
    u = mix32_t(seed, 21, i, z)
    if skew:
        u2 = mix32_t(seed, 22, i, z)
        v = ((u % n_values) * (u2 % n_values)) // max(1, n_values)
    else:
        v = u % n_values
    hi = mix32_t(seed, 23, v, z)
    lo = mix32_t(seed, 24, v, z)
    return ((hi - (1 << 31)) << 32) | lo
