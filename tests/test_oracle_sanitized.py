"""The oracle under AddressSanitizer + UndefinedBehaviorSanitizer: every
entry point of oracle/oracle_cd.c is driven once, with ragged sizes and the edge cases of the
method (n = 0, accepted slots, all -inf rows, LIMIT, row_map, padded strides), in a child process
that preloads gcc's libasan and loads oracle/liboracle_cd_san.so.  Any out-of-bounds access,
use-after-free, signed overflow or misaligned access aborts the child."""
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

SCRIPT = r"""
import numpy as np, torch
import oracle, workloads as wl
assert oracle.oracle_cd._load()._name.endswith("liboracle_cd_san.so")
cfg = wl.scaled(wl.CONFIGS["c3"], V=1000, B=37, S=11, max_steps=5)
aut = wl.build_automaton(cfg)
assert oracle.validate(aut) == 0
x = wl.build_step_logits(cfg, aut)
live = [s for s in range(aut.S) if not aut.accepting[s]]
acc = [s for s in range(aut.S) if aut.accepting[s]]
states = [live[i % len(live)] if i % 4 else (acc[0] if acc else live[0]) for i in range(cfg.B)]
perm = np.random.default_rng(0).permutation(cfg.B)
tok, lp, lse, done, st = oracle.step(aut, x[0], states, row_map=perm)
oracle.step(aut, x[0][:0], [])
y = x[0].float().clone(); y[:] = float("-inf"); oracle.step(aut, y, [live[0]] * cfg.B)
oracle.compact(done, perm, st); oracle.compact(np.zeros(0, np.uint8))
oracle.decode_loop(aut, x)
sat = (aut.accepting.numpy() * (np.arange(aut.S) % 2 == 0)).astype(np.uint8)
oracle.decode_loop(aut, x, satisfying=sat, limit=3)
oracle.sample_step(aut, x[0], states, 0.7, seed=5, step=2, row_map=perm)
oracle.sample_decode_loop(aut, x, 1.3, seed=9)
H = 24
W = wl.make_head(1, cfg.V, H, 2.0, ld=32); hid = [wl.make_hidden(1, k, cfg.B, H, ld=40) for k in range(3)]
oracle.head_step(aut, hid[0], W, H, states, row_map=perm)
oracle.head_decode_loop(aut, hid, W, H)
keys = wl.make_keys(3, 500, 17, skew=True)
rep, dr = oracle.dedup(keys)
res = dict(tokens=np.zeros((len(dr), 3), np.int32), len=np.zeros(len(dr), np.int32), final_state=np.zeros(len(dr), np.int32),
           sum_logprob=np.zeros(len(dr)), done=np.ones(len(dr), np.uint8))
oracle.join_results(rep, res)
oracle.filter_rows(np.arange(40) % aut.S, np.ones(40, np.uint8), sat)
oracle.det_logf(0.3); oracle.gumbel(1, 2, 3, 4)
print("sanitized oracle ok")
"""


def test_oracle_runs_clean_under_asan_and_ubsan():
    import oracle

    oracle.build(sanitize=True)
    env = dict(os.environ)
    env.update(LD_PRELOAD=oracle.asan_runtime(), ORACLE_CD_SANITIZE="1", PYTHONPATH=ROOT,
               ASAN_OPTIONS="detect_leaks=0:halt_on_error=1:abort_on_error=0",
               UBSAN_OPTIONS="halt_on_error=1:print_stacktrace=1")
    p = subprocess.run([sys.executable, "-c", SCRIPT], cwd=ROOT, env=env, capture_output=True, text=True, timeout=600)
    assert p.returncode == 0, p.stderr[-3000:]
    assert "sanitized oracle ok" in p.stdout
    assert "AddressSanitizer" not in p.stderr and "runtime error" not in p.stderr, p.stderr[-3000:]
