"""Automata of typed outputs, written out as definitions -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

O11 (SURVEY.md 8(c) G4 / G5, 8(f) N5 second half): the EOS / longest-match variant of "when is a
row finished".  The paper restricts a generation to the strings of an `options` set or a quantified
collection (section 2.3) and leaves the stopping rule to the engine (L226: the
decoding rule is open; llguidance / vLLM arbitrate through EOS, L183, L204).  Reading (G4): the
language of an option set with an end-of-sequence token is

    L = { label + [eos] : label in labels }

so a label that is a token-prefix of another label ("New York" / "New York City") is fine: in the
state reached by the shorter label the model either emits eos (stop: the shorter label) or goes on
(longest match is the model's choice, token by token).  "Every may-stop state gets an eos edge to
one accepting sink; only the sink accepts."

The automaton of a finite language is its prefix tree -- that is all this file builds.  It shares
nothing with paper_2606_31808_b200/ (whose builder is csrc/cd_types.hpp) and must never be imported
from it.  Pure-python loops: option sets are small.

State numbering (the convention the product's C-ABI header documents for its option-set sugar with eos >= 0, so that
final states compare bit for bit): state 0 is the empty prefix; the other proper prefixes of L are
numbered in order of first appearance when the strings are inserted in the given order, token by
token; the single accepting sink is numbered last (S - 1).

Pins: tests/test_oracle_eos_pins.py (a hand-written CSR for {"a", "a b"}, the language enumerated by
DFS, decoding by hand from four logits, rejections, agreement with the leaf-per-label trie on
prefix-free sets).
"""
from __future__ import annotations

from typing import Dict, List, Sequence, Tuple

import numpy as np


class TypeAutomaton:
    """Host CSR image (the argument list of cd_compile_dfa / what oracle.decode_loop takes)."""

    def __init__(self, V, S, start, row_ptr, tok, next, accepting):
        self.V, self.S, self.start = int(V), int(S), int(start)
        self.row_ptr = np.asarray(row_ptr, np.int64)
        self.tok = np.asarray(tok, np.int32)
        self.next = np.asarray(next, np.int32)
        self.accepting = np.asarray(accepting, np.uint8)

    @property
    def nnz(self) -> int:
        return int(self.tok.shape[0])


def language_dfa(V: int, strings: Sequence[Sequence[int]]) -> TypeAutomaton:
    """The prefix-tree automaton of a finite language under "a row is finished the first time its
    state accepts" (G4): every proper prefix of a string is a state, every complete string leads to
    the one accepting sink.  For every string to be reachable the language must be prefix-free
    (no string a proper prefix of another) and duplicate-free; both are checked."""
    if V < 1:
        raise ValueError("V must be >= 1")
    strings = [tuple(int(t) for t in s) for s in strings]
    if not strings:
        raise ValueError("empty language")
    if len(set(strings)) != len(strings):
        raise ValueError("duplicate string")
    for s in strings:
        if len(s) == 0:
            raise ValueError("empty string")
        if any(t < 0 or t >= V for t in s):
            raise ValueError("token outside [0, V)")
    whole = set(strings)
    state_of: Dict[Tuple[int, ...], int] = {(): 0}  # proper prefix -> state id, in order of first appearance
    for s in strings:
        for j in range(1, len(s)):
            p = s[:j]
            if p in whole:
                raise ValueError("language is not prefix-free")
            if p not in state_of:
                state_of[p] = len(state_of)
    sink = len(state_of)
    edges: List[Dict[int, int]] = [dict() for _ in range(sink + 1)]
    for s in strings:
        edges[state_of[s[:-1]]][s[-1]] = sink
        for j in range(1, len(s)):
            edges[state_of[s[: j - 1]]][s[j - 1]] = state_of[s[:j]]
    row_ptr, tok, nxt = [0], [], []
    for e in edges:
        for t in sorted(e):
            tok.append(t)
            nxt.append(e[t])
        row_ptr.append(len(tok))
    accepting = [0] * sink + [1]
    return TypeAutomaton(V, sink + 1, 0, row_ptr, tok, nxt, accepting)


def trie_eos(V: int, labels: Sequence[Sequence[int]], eos: int) -> TypeAutomaton:
    """O11: the option set `labels` with end-of-sequence token `eos`: L = { label + [eos] }.  Labels
    must be non-empty, distinct and must not contain eos (then L is prefix-free whatever the prefix
    relations among the labels themselves)."""
    if not (0 <= eos < V):
        raise ValueError("eos outside [0, V)")
    labs = [tuple(int(t) for t in l) for l in labels]
    for l in labs:
        if len(l) == 0:
            raise ValueError("empty label")
        if eos in l:
            raise ValueError("label contains eos")
    if len(set(labs)) != len(labs):
        raise ValueError("duplicate label")
    return language_dfa(V, [l + (eos,) for l in labs])


def list_language(labels: Sequence[Sequence[int]], open_: Sequence[int], sep: Sequence[int], close: Sequence[int],
                  min_items: int, max_items: int, eos: int = -1) -> List[Tuple[int, ...]]:
    """The strings of a collection type with a quantifier ("{3} for exactly three, {1,5}
    for between one and five"):  open item (sep item)^(c-1) close [eos]  for min_items <= c <= max_items,
    every item one of `labels`.  Written out with nested loops; duplicates (two item sequences spelling
    the same token string) are kept so that the caller sees the ambiguity."""
    out: List[Tuple[int, ...]] = []

    def rec(prefix: Tuple[int, ...], count: int):
        if min_items <= count <= max_items:
            out.append(prefix + tuple(close) + ((eos,) if eos >= 0 else ()))
        if count == max_items:
            return
        for lab in labels:
            rec(prefix + (tuple(sep) if count > 0 else ()) + tuple(lab), count + 1)

    rec(tuple(open_), 0)
    return out
