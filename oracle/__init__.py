"""CPU oracle for the constrained-decoding step -- TEST INFRASTRUCTURE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs may import this package.  See oracle_cd.c.
"""
from .oracle_cd import (  # noqa: F401
    OracleError,
    asan_runtime,
    build,
    compact,
    decode_loop,
    dedup,
    det_logf,
    gumbel,
    fmix32,
    sample_decode_loop,
    sample_step,
    filter_rows,
    join_results,
    head_decode_loop,
    head_logit,
    head_step,
    step,
    validate,
)
from .oracle_types import TypeAutomaton, language_dfa, list_language, trie_eos  # noqa: F401
