"""B200-native batched type-constrained decoding step (arxiv/paper_2606_31808 hot path).

Thin Python binding over the C-ABI library libcd.so (include/cd.h): argument
marshalling only, every step of the path runs in the CUDA kernels under
csrc/.  PyTorch is used for device memory and streams, nothing else.  There is
no CPU fallback: if libcd.so is missing or no CUDA device is present the calls
raise.
"""
from .binding import (  # noqa: F401
    BF16,
    F32,
    LOOP_AUTO,
    LOOP_BARRIER,
    LOOP_PER_STEP,
    build_trie,
    CdError,
    Dfa,
    compact,
    compact_noalloc,
    COMPACT_NOALLOC_MAX_N,
    build_list,
    compile_dfa,
    compile_list,
    compile_trie,
    decode_loop,
    decode_loop_async,
    loop_sync,
    PreparedLoop,
    decode_loop_cb,
    head_decode_loop_cb,
    decode_loop_host,
    dedup,
    filter_rows,
    join_results,
    head_decode_loop,
    head_decode_loop_host,
    head_step,
    launch_count,
    probe_read,
    lib,
    lib_path,
    step,
    transition,
)
