#!/usr/bin/env python
"""bench.py -- constrained-step throughput on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config c4] [--impl reference]

A "step" is one pass of the whole hot path over one batch of synthetic input:
cd_decode_loop on one batch of the workload (automaton store already
compiled): per decoding step the fused mask + masked log-softmax + masked
argmax + CSR transition kernel, then early-exit compaction, until max_steps.
Default workload: one batch of BASELINE.json configs[4] (B=4096 rows,
V=262144, bf16, random DFA S=4096 at 0.5 % density, <= 16 steps, 32 GiB of
logits per batch) -- the largest single-GPU configuration.  `value` is table
rows/s (rows decoded to completion or truncation per second, all GPUs).

Prints ONE JSON line (rank 0).  See DESIGN.md "Measurement" for every field.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import torch  # noqa: E402

import workloads as wl  # noqa: E402

METRIC = "constrained-step rows/s and HBM GB/s (% of B200 peak) at V=262144"
UNIT = "rows/s"
NOMINAL_HBM_GBS = 8000.0
FALLBACK_HBM_GBS = 6650.0  # /opt/skills/guides/B200_PROFILING.md fallback
FALLBACK_BF16_TFLOPS = 1590.0  # /opt/skills/guides/B200_PROFILING.md fallback
READ_RATE_GBS = 7200.0  # the kernel's own pure-read probe on this pool (cd_probe_read): used for the fixed-cost estimate only


def ncu_traffic(kernel: str, config: str):
    """dram__bytes_read.sum + dram__bytes_write.sum of ONE launch of `kernel` on `config` from the committed
    `ncu --set full` captures, listed in profiles/ncu_traffic.csv (kernel,config,dram_read_bytes,
    dram_write_bytes,profile,note).  Not measured in this run (never profile a timed run): the JSON names
    the capture it comes from; None if no capture of that kernel / config is committed."""
    path = os.path.join(ROOT, "profiles", "ncu_traffic.csv")
    try:
        for line in open(path):
            p = [x.strip() for x in line.split(",")]
            if len(p) >= 5 and p[0] == kernel and p[1] == config:
                return {"bytes": int(p[2]) + int(p[3]), "profile": p[4]}
    except Exception:
        pass
    return None


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="c4", choices=["c1", "c2", "c3", "c4"])
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--batches", type=int, default=2, help="resident input batches rotated over the timed steps")
    ap.add_argument("--cpu-sample-rows", type=int, default=512)
    ap.add_argument("--gather-max", type=int, default=0,
                    help="cd_set_gather_max for the main measurement: 0 = dense scan (default, the graded method), "
                         "-1 = automatic, > 0 = threshold (SURVEY 8(f) N1)")
    ap.add_argument("--no-adaptive", action="store_true", help="skip the density-adaptive (gather) measurement")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-dedup", action="store_true", help="skip the early-deduplication measurement (SURVEY 8(f) N4)")
    ap.add_argument("--no-head", action="store_true", help="skip the LM-head fused step measurement (SURVEY 8(f) N2)")
    ap.add_argument("--head-H", type=int, default=2560, help="hidden size of the LM head (Gemma 3 4B: 2560)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--verbose", action="store_true", help="per-launch table of the step kernel on stderr")
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"],
                    help="weak: every rank decodes its own batches (default); strong: ONE batch of B rows is "
                         "sharded B/N rows per rank (SURVEY 8(e): contiguous row ranges, no collective)")
    ap.add_argument("--no-per-config", action="store_true", help="skip the c1-c3 block (per_config)")
    ap.add_argument("--loop-mode", default="auto", choices=["auto", "barrier", "per_step"],
                    help="auto: cd_decode_loop as ONE persistent kernel, every row advancing on its own (default); "
                         "barrier: the lock-step persistent kernel; per_step: one launch per decoding step")
    return ap.parse_args()


def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region."""

    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.proc = None
        self.path = None

    def start(self):
        try:
            fd, self.path = tempfile.mkstemp(suffix=".csv")
            os.close(fd)
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "100",
                 "-i", str(self.index)],
                stdout=open(self.path, "w"), stderr=subprocess.DEVNULL)
            time.sleep(0.35)
        except Exception:
            self.proc = None

    def stop(self):
        if self.proc is None:
            return None
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        try:
            for line in open(self.path):
                p = [x.strip() for x in line.split(",")]
                if len(p) < 9:
                    continue
                try:
                    sm.append(float(p[1]))
                    mx.append(float(p[2]))
                except ValueError:
                    continue
                for nm, v in zip(names, p[5:9]):
                    if v.lower().startswith("active"):
                        reasons.add(nm)
            os.unlink(self.path)
        except Exception:
            return None
        if not sm:
            return None
        return {"sm_mhz": statistics.median(sm), "sm_max_mhz": max(mx), "reasons": sorted(reasons),
                "samples": len(sm)}


def measured_tensor_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            j = json.load(open(p))
            return float(j["bf16_tflops"]), float(j.get("bf16_tflops_sustained", j["bf16_tflops"])), \
                "measured (MEASURED_PEAKS.json bf16_tflops, burst)"
        except Exception:
            pass
    return FALLBACK_BF16_TFLOPS, FALLBACK_BF16_TFLOPS, "fallback (B200_PROFILING.md)"


def head_section(cd, cfg, aut, dfa, device, H, iters, warmup):
    """one constrained step fused with the LM head (cd_head_step) for B rows spread
    over the automaton's live states (the state mix of a mid-loop step), W [V, H] bf16 ~ N(0, 2/sqrt(H)),
    hidden ~ N(0,1).  W (1.34 GB at H=2560) is larger than L2, so every call streams it from HBM.
    The dominant kernel is the tcgen05 contraction (bound: tensor); its algorithmic flops are
    2 * n_dense * V * H per call.  The unfused alternative (library GEMM writing bf16 logits, then
    cd_step reading them) is timed beside it."""
    V, n = cfg.V, cfg.B
    stream = torch.cuda.current_stream()
    W = wl.make_head(7, V, H, 2.0, device=device)
    hid = wl.make_hidden(cfg.seed, 0, n, H, device=device)
    acc = torch.as_tensor(aut.accepting)
    live = torch.nonzero(acc == 0).flatten().to(torch.int32)
    st0 = live[(torch.arange(n) * 7) % live.numel()].to(device) if cfg.kind == "dfa" else \
        torch.zeros(n, dtype=torch.int32, device=device)
    st = st0.clone()
    i32 = dict(dtype=torch.int32, device=device)
    outb = (torch.empty(n, **i32), torch.empty(n, dtype=torch.float32, device=device),
            torch.empty(n, dtype=torch.float32, device=device), torch.empty(n, dtype=torch.uint8, device=device))
    deg = torch.diff(torch.as_tensor(aut.row_ptr))
    auto_max = max(1, V // 300)  # the library's automatic threshold (cd_api.cu head_gather_max_for)
    n_dense = int((deg[st0.cpu().long()] > auto_max).sum())

    def timed(fn):
        for _ in range(warmup):
            fn()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(iters):
            fn()
        e1.record(stream)
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / iters

    def fused():
        st.copy_(st0)
        cd.head_step(dfa, hid, W, st, out=outb)

    l0 = cd.launch_count()
    ms_f = timed(fused)
    launches = (cd.launch_count() - l0) // (iters + warmup)
    tok_f = outb[0].clone()
    logits = torch.empty((n, V), dtype=torch.bfloat16, device=device)

    def unfused():
        st.copy_(st0)
        torch.matmul(hid, W.t(), out=logits)
        cd.step(dfa, logits, st, out=outb)

    ms_u = timed(unfused)
    agree = float((tok_f == outb[0]).float().mean())  # bf16 rounding of the logits may flip near-ties
    ms_g = timed(lambda: torch.matmul(hid, W.t(), out=logits))
    del logits
    # the whole decode loop on the head path: table rows/s (the bench's metric), device-resident hidden
    # states and end to end from pinned host hidden states (H2D of every step's [B, H] inside the timed
    # region, results read back to the host)
    dfa.set_sampling(0.0)
    hs_dev = [wl.make_hidden(cfg.seed, k, n, H, device=device) for k in range(cfg.max_steps)]
    lout = None

    def loop_dev():
        nonlocal lout
        lout = cd.head_decode_loop(dfa, hs_dev, W, H=H, out=lout)

    ms_loop = timed(loop_dev)
    row_steps_loop = int(lout["len"].sum())
    hs_host = [h.cpu().pin_memory() for h in hs_dev]
    hout = None
    cd.head_decode_loop_host(dfa, hs_host, W, H=H)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    k_e2e = 3
    for _ in range(k_e2e):
        hout = cd.head_decode_loop_host(dfa, hs_host, W, H=H, out=hout)
    torch.cuda.synchronize()
    dt_e2e = (time.perf_counter() - t0) / k_e2e
    assert torch.equal(hout["tokens"], lout["tokens"].cpu()), "host-buffer head loop disagrees with the device loop"
    loop = {"value": n / (ms_loop * 1e-3), "unit": UNIT, "ms_per_step": ms_loop, "row_steps_per_loop": row_steps_loop,
            "e2e": {"value": n / dt_e2e, "unit": UNIT, "ms_per_step": 1e3 * dt_e2e,
                    "h2d_bytes_per_step": cfg.max_steps * n * H * 2,
                    "d2h_bytes_per_step": n * (cfg.max_steps * 4 + 13), "host_memory": "pinned"},
            "note": "one step = cd_head_decode_loop over one batch of B rows (all max_steps steps); the model forward that "
                    "produces the hidden states is outside the path"}
    del hs_dev, hs_host
    burst, sustained, src = measured_tensor_peak()
    flops = 2.0 * n_dense * V * H
    ach = flops / (ms_f * 1e-3) / 1e12 if n_dense else 0.0
    if n_dense == 0:
        # every row gathered: the call reads deg W rows of 2H bytes per row (mostly from L2: rows in
        # the same state share them) -- no dense contraction, no tensor roofline
        gbytes = float(deg[st0.cpu().long()].sum()) * 2 * H
        roof = {"bound": "hbm", "kernel": "cd::head_gather_kernel (gathered dot products through the CSR token list)",
                "achieved": gbytes / (ms_f * 1e-3) / 1e9, "peak": measured_peak()[0], "unit": "GB/s",
                "frac": gbytes / (ms_f * 1e-3) / 1e9 / measured_peak()[0], "traffic": None,
                "note": "bytes = W rows touched (2H each), served by L2 when rows share a state; launch-latency bound at this size"}
    else:
        roof = None
    hk = "cd::head_dense2_kernel" if n_dense > 128 else "cd::head_dense_kernel"  # which kernel ran the contraction
    head = {
        "workload": f"{cfg.name}: one cd_head_step, n={n} rows over the live states, V={V}, H={H} bf16 "
                    f"(Gemma 3 4B head shape, PAPER.md L191), {n_dense} rows dense / {n - n_dense} gathered",
        "ms_per_step": ms_f, "row_steps_per_s": n / (ms_f * 1e-3), "gpu_launches_per_step": int(launches),
        "decode_loop": loop,
        "unfused_ms_per_step": ms_u, "library_gemm_ms": ms_g, "speedup_vs_unfused": ms_u / ms_f,
        "token_agreement_with_unfused_bf16_logits": agree,
        "roofline": roof or {"bound": "tensor", "kernel": hk + (" (CTA pairs: tcgen05 cta_group::2 256x256x16, 6-stage TMA ring, masked online-softmax epilogue from TMEM)"
                                                               if n_dense > 128 else " (tcgen05 128x256x16, masked online-softmax epilogue from TMEM)"),
                     "achieved": ach, "peak": burst, "unit": "TFLOP/s", "frac": ach / burst if burst else None,
                     "peak_source": src, "frac_of_sustained_peak": ach / sustained if sustained else None,
                     "frac_of_nominal_2250": ach / 2250.0, "flops_per_launch": flops,
                     "note": "timed over the whole call (prepare + pack + contraction + finish), so the kernel's own rate is higher",
                     "traffic": (ncu_traffic(hk, cfg.name) or {}).get("bytes"),
                     "traffic_source": (ncu_traffic(hk, cfg.name) or {}).get("profile")},
    }
    return head


def dedup_section(cd, device, iters, warmup):
    """SELECT DISTINCT + LEFT JOIN as device primitives on a table of
    N = 2^20 row keys with 4096 distinct values (duplication factor 256, long-tailed).  Reports rows/s of
    cd_dedup and cd_join_results; algorithmic bytes: dedup reads 8 B and writes 4 B per row (+ the distinct
    list), join reads 4 B and writes (max_steps + 3) * 4 + 1 B per row."""
    N, nv, ms_steps = 1 << 20, 4096, 16
    stream = torch.cuda.current_stream()
    keys = wl.make_keys(4, N, nv, device=device, skew=True)
    out = (torch.empty(N, dtype=torch.int32, device=device), torch.empty(N, dtype=torch.int32, device=device),
           torch.empty(1, dtype=torch.int32, device=device))

    def timed(fn):
        for _ in range(warmup):
            fn()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(iters):
            fn()
        e1.record(stream)
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / iters

    ms_d = timed(lambda: cd.dedup(keys, out=out))
    rep, dr, nd = cd.dedup(keys, out=out)
    D = int(nd)
    i32 = dict(dtype=torch.int32, device=device)
    res_d = dict(tokens=torch.zeros((D, ms_steps), **i32), len=torch.zeros(D, **i32), final_state=torch.zeros(D, **i32),
                 sum_logprob=torch.zeros(D, dtype=torch.float32, device=device),
                 done=torch.zeros(D, dtype=torch.uint8, device=device))
    jout = cd.join_results(rep, res_d)
    ms_j = timed(lambda: cd.join_results(rep, res_d, out=jout))
    peak = measured_peak()[0]
    b_d = N * 12 + D * 4
    b_j = N * (4 + (ms_steps + 3) * 4 + 1)
    return {"workload": f"N={N} row keys, {D} distinct values (duplication factor {N / D:.0f}, long-tailed), max_steps={ms_steps}",
            "dedup_ms": ms_d, "dedup_rows_per_s": N / (ms_d * 1e-3), "dedup_gbs": b_d / (ms_d * 1e-3) / 1e9,
            "join_ms": ms_j, "join_rows_per_s": N / (ms_j * 1e-3), "join_gbs": b_j / (ms_j * 1e-3) / 1e9,
            "join_frac_of_hbm_peak": b_j / (ms_j * 1e-3) / 1e9 / peak,
            "lm_calls_saved": f"{N - D} of {N} generations (factor {N / D:.0f})",
            "note": "dedup is bound by hash-table atomics (2 per key onto few hot words: profiles/r3a_dedup_join.md), not by bytes; both are "
                    "negligible next to the decode loop they remove (256 batches x ~4 ms)"}


def build_inputs(cfg, device, n_batches, batch0, rows=None):
    aut = wl.build_automaton(cfg, device=device)
    batches = [wl.build_step_logits(cfg, aut, device=device, batch=batch0 + b, rows=rows) for b in range(n_batches)]
    return aut, batches


def bytes_per_row_step(cfg):
    sz = 2 if cfg.dtype == torch.bfloat16 else 4
    return cfg.V * sz, cfg.V // 8


def replay_stepwise(cd, cfg, aut, dfa, logits, device, timed):
    """One decode loop of `logits` driven through the stepwise API (cd_step + cd_compact) with the active
    count read back after every step: gives, per decoding step, the active rows n_k, the number of
    distinct automaton states among them (each costs one 32 KiB mask row from HBM) and the
    sum of their out-degrees.  timed=True replays it once more with everything enqueued ahead of the GPU
    (a device-side sleep first, no host sync, preallocated outputs) and a CUDA event pair around every
    cd_step launch, so that the events bracket the kernel itself and not the host's launch gaps."""
    stream = torch.cuda.current_stream()
    B = logits[0].shape[0]
    i32 = dict(dtype=torch.int32, device=device)
    deg_dev = torch.diff(torch.as_tensor(aut.row_ptr)).to(device)
    bufs = dict(tok=torch.empty(B, **i32), lp=torch.empty(B, dtype=torch.float32, device=device),
                done=torch.empty(B, dtype=torch.uint8, device=device),
                ids=[torch.empty(B, **i32) for _ in range(2)], st=[torch.empty(B, **i32) for _ in range(2)],
                na=torch.empty(1, **i32))
    n_k, distinct_k, deg_k, step_ms = [], [], [], []
    for rep in range(2 if timed else 1):
        bufs["ids"][0].copy_(torch.arange(B, **i32))
        bufs["st"][0].fill_(aut.start)
        events = []
        if rep == 1:
            torch.cuda.synchronize()
            torch.cuda._sleep(600000)
        n = B
        for k in range(cfg.max_steps):
            cur, nxt = k & 1, (k + 1) & 1
            if rep == 0:
                if n == 0:
                    break
                n_k.append(n)
                distinct_k.append(int(torch.unique(bufs["st"][cur][:n]).numel()))
                deg_k.append(int(deg_dev[bufs["st"][cur][:n].long()].sum()))
            elif k >= len(n_k):
                break
            else:
                n = n_k[k]
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(stream)
            cd.step(dfa, logits[k], bufs["st"][cur], row_map=bufs["ids"][cur], n=n, want_lse=False,
                    out=(bufs["tok"], bufs["lp"], None, bufs["done"]))
            b.record(stream)
            events.append((a, b))
            cd.compact(bufs["done"], bufs["ids"][cur], bufs["st"][cur], n=n,
                       out=(bufs["ids"][nxt], bufs["st"][nxt], bufs["na"]))
            if rep == 0:
                n = int(bufs["na"])
        torch.cuda.synchronize()
        if rep == 1:
            step_ms = [a.elapsed_time(b) for a, b in events]
    return n_k, distinct_k, deg_k, step_ms


def measure_loop(cd, cfg, aut, dfa, batches, device, steps, warmup, peak, verbose=False, label="", pipelined=True):
    """The decode loop of one configuration: K timed cd_decode_loop calls over the rotated resident
    batches (CUDA events on the launching stream), then the per-step picture of the persistent kernel
    from its own device-side trace (cd_loop_trace: active rows and nanoseconds per decoding step) with
    the algorithmic bytes of every step (n_k logits rows + one mask row per distinct state)."""
    stream = torch.cuda.current_stream()
    sz_logit, sz_mask = bytes_per_row_step(cfg)
    out = None
    per_batch = []
    for b, logits in enumerate(batches):  # untimed: per-step n_k / distinct states / bytes of every resident batch
        n_k, distinct_k, deg_k, _ = replay_stepwise(cd, cfg, aut, dfa, logits, device, timed=False)
        per_batch.append(dict(n=n_k, distinct=distinct_k, deg=deg_k,
                              bytes=[n * sz_logit + d * sz_mask for n, d in zip(n_k, distinct_k)]))
    # the K loops are enqueued back to back (cd_decode_loop_async: one kernel launch each, arguments marshalled once
    # per resident batch, every batch its own output buffers) and the stream is synchronised once at the end
    # (cd_loop_sync, which also reports the device-side status of all K loops)
    # (pipelined=False: cd_decode_loop, which synchronises the stream after every loop -- the lock-step kernel
    # holds the device's cooperative-launch lock until it has finished and has no asynchronous form)
    loops = [cd.PreparedLoop(dfa, b, max_steps=cfg.max_steps) for b in batches]
    go = (lambda lp: lp.enqueue()) if pipelined else (lambda lp: lp.run())
    for i in range(warmup):
        go(loops[i % len(loops)])
    loops[0].sync()
    l0 = cd.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for i in range(steps):
        go(loops[(warmup + i) % len(loops)])
    e1.record(stream)
    loops[0].sync()
    out = loops[(warmup + steps - 1) % len(loops)].out
    launches = cd.launch_count() - l0
    ms = e0.elapsed_time(e1) / steps
    timed = [(warmup + i) % len(batches) for i in range(steps)]
    loop_bytes = sum(sum(per_batch[b]["bytes"]) for b in timed) / steps
    row_steps = sum(sum(per_batch[b]["n"]) for b in timed) / steps
    # the last timed loop, step by step, from the kernel's own trace
    last = per_batch[timed[-1]]
    tr_n, tr_ns = dfa.loop_trace()
    res = {
        "B": cfg.B, "max_steps": cfg.max_steps, "resident_batches": len(batches), "loops_timed": steps,
        "loops_enqueued": "back to back (cd_decode_loop_async), one cd_loop_sync at the end" if pipelined else "cd_decode_loop (stream synchronised after every loop)",
        "rows_per_s": cfg.B / (ms * 1e-3), "ms_per_loop": ms, "row_steps_per_loop": row_steps,
        "gpu_launches_per_loop": launches / steps,
        "loop_gbs": loop_bytes / (ms * 1e-3) / 1e9,
        "frac_of_measured_peak": loop_bytes / (ms * 1e-3) / 1e9 / peak,
        "frac_of_nominal_8TBs": loop_bytes / (ms * 1e-3) / 1e9 / NOMINAL_HBM_GBS,
        "bytes_per_loop": loop_bytes,
        "n_per_step": last["n"],
    }
    if tr_n and tr_n == last["n"]:
        us = [t / 1e3 for t in tr_ns]
        gbs = [b / (max(t, 1) * 1e-9) / 1e9 for b, t in zip(last["bytes"], tr_ns)]  # (the device timer ticks every 256 ns)
        fixed = [u - b / (READ_RATE_GBS * 1e3) for u, b in zip(us, last["bytes"])]
        kern_us = sum(us)
        k0 = max(range(len(us)), key=lambda k: last["bytes"][k])
        res.update({
            "kernel": "cd::flow_kernel (one launch per loop; every row advances on its own, no grid barrier)",
            "kernel_us_per_loop": kern_us,
            "kernel_gbs": sum(last["bytes"]) / (kern_us * 1e-6) / 1e9,
            "kernel_frac_of_measured_peak": sum(last["bytes"]) / (kern_us * 1e-6) / 1e9 / peak,
            "kernel_frac_of_nominal_8TBs": sum(last["bytes"]) / (kern_us * 1e-6) / 1e9 / NOMINAL_HBM_GBS,
            "largest_step": {"n": last["n"][k0], "us": us[k0], "gbs": gbs[k0], "frac_of_measured_peak": gbs[k0] / peak,
                             "frac_of_nominal_8TBs": gbs[k0] / NOMINAL_HBM_GBS},
            "us_per_step": [round(u, 2) for u in us],
            "gbs_per_step": [round(g, 0) for g in gbs],
            "fixed_us_per_step_avg": sum(fixed) / len(fixed),
            "fixed_cost_note": f"step time minus its bytes at the kernel's pure-read rate ({READ_RATE_GBS:.0f} GB/s); rows advance on "
                               "their own: a step lasts from the last publication of a row's step k to that of a row's step k + 1, so "
                               "the first step carries the pipeline fill and single steps can come out below their byte time",
        })
        if verbose:
            for k, (n, u, g, f) in enumerate(zip(last["n"], us, gbs, fixed)):
                print(f"  {label} step {k:2d}: n={n:5d} distinct={last['distinct'][k]:5d} {u:8.1f} us {g:7.0f} GB/s "
                      f"fixed {f:5.1f} us", file=sys.stderr)
    else:
        res["kernel"] = "cd::step_kernel (one launch per decoding step)"
    return res, per_batch, out


def per_config_section(cd, device, peak, verbose):
    """BASELINE.json configs c1-c3 beside the c4 headline (north_star: "on all five configs", ">= 70 % ... at
    V = 262144, B >= 1024" covers c2): the same event protocol; 4 resident batches for c1 / c2 and 2 for c3 (a
    loop streams 0.27 / 1.9 / 2.7 GB of distinct logits, all larger than the 126 MB L2, and consecutive loops
    use different batches)."""
    out = {}
    for name, nb, k in (("c1", 4, 40), ("c2", 4, 20), ("c3", 2, 10)):
        cfg = wl.CONFIGS[name]
        aut, batches = build_inputs(cfg, device, nb, 0)
        dfa = cd.compile_dfa(aut.V, aut.S, aut.start, aut.row_ptr, aut.tok, aut.next, aut.accepting, device=device)
        dfa.reserve(cfg.B)
        res, _, _ = measure_loop(cd, cfg, aut, dfa, batches, device, k, 5, peak, verbose=verbose, label=name)
        sy, _, _ = measure_loop(cd, cfg, aut, dfa, batches, device, k, 5, peak, pipelined=False)
        res["sync_after_every_loop"] = {"rows_per_s": sy["rows_per_s"], "ms_per_loop": sy["ms_per_loop"],
                                        "frac_of_measured_peak": sy["frac_of_measured_peak"]}
        # the same loops as one launch per decoding step (the round-1 structure; still what the callback / host
        # forms use) and in the lock-step persistent kernel (grid barrier per step; what a LIMIT loop runs in)
        dfa.set_loop_mode(cd.LOOP_PER_STEP)
        ps, _, _ = measure_loop(cd, cfg, aut, dfa, batches, device, k, 5, peak)
        res["per_step_launches"] = {"rows_per_s": ps["rows_per_s"], "ms_per_loop": ps["ms_per_loop"], "loop_gbs": ps["loop_gbs"],
                                    "frac_of_measured_peak": ps["frac_of_measured_peak"]}
        dfa.set_loop_mode(cd.LOOP_BARRIER)
        lb, _, _ = measure_loop(cd, cfg, aut, dfa, batches, device, k, 5, peak, pipelined=False)
        res["lock_step_kernel"] = {"rows_per_s": lb["rows_per_s"], "ms_per_loop": lb["ms_per_loop"],
                                   "kernel_us_per_loop": lb.get("kernel_us_per_loop"), "kernel_gbs": lb.get("kernel_gbs"),
                                   "us_per_step": lb.get("us_per_step"), "fixed_us_per_step_avg": lb.get("fixed_us_per_step_avg")}
        dfa.set_loop_mode(cd.LOOP_AUTO)
        # density-adaptive (tries never need the scan)
        dfa.set_gather_max(-1)
        ga, _, _ = measure_loop(cd, cfg, aut, dfa, batches, device, k, 5, peak)
        res["adaptive_rows_per_s"] = ga["rows_per_s"]
        dfa.close()
        del batches
        torch.cuda.empty_cache()
        res["workload"] = cfg.desc
        out[name] = res
    return out


def run_reference(args, rank):
    """--impl reference: the CPU oracle, as it stands, timed on this box's host
    cores on a bounded sample (the first --cpu-sample-rows rows of each batch)."""
    if rank != 0:
        return
    import oracle

    oracle.build()
    cfg = wl.CONFIGS[args.config]
    R = min(args.cpu_sample_rows, cfg.B)
    dev = "cuda:0" if torch.cuda.is_available() else "cpu"
    aut = wl.build_automaton(cfg, device=dev)
    # the sample: rows [0, R) of every step buffer of batch 0 (generated on `dev`, bytes moved to the host)
    # (make_logits draws rows in chunks of 512 from one generator stream, so the first chunks of a
    # smaller batch are byte-identical to those of the full batch)
    gen_rows = min(cfg.B, (R + 511) // 512 * 512)
    logits = [x[:R].cpu().contiguous() for x in wl.build_step_logits(cfg, aut, device=dev, B=gen_rows)]
    times, row_steps = [], 0
    for i in range(args.warmup + args.steps):
        t0 = time.perf_counter()
        res = oracle.decode_loop(aut, logits)
        dt = time.perf_counter() - t0
        if i >= args.warmup:
            times.append(dt)
            row_steps = int(res["n_active_hist"].sum())
    total = sum(times)
    value = R * args.steps / total
    sample = f"rows [0,{R}) of one {cfg.name} batch (B={cfg.B}), all {cfg.max_steps} steps, {row_steps} row-steps per pass"
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * total / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "logits_dtype": str(cfg.dtype).replace("torch.", ""),
        "data": "synthetic", "config": {"workload": cfg.desc, "sample": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "host_cores": os.cpu_count(), "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "row_steps_per_s": row_steps * args.steps / total,
    }
    print(json.dumps(line), flush=True)


def launcher_command(args_gpus: int, argv, master_port: int = 0):
    """`python bench.py --gpus N` with N > 1 outside torchrun: the command that starts N ranks of this same
    script on this node (one rank per GPU over NCCL; rendezvous on 127.0.0.1, the hostname may not resolve)."""
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args_gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(master_port or 29500 + os.getpid() % 2000)]
    return cmd + [os.path.abspath(__file__)] + list(argv)


def check_gpus(requested: int, visible: int):
    """A request for more GPUs than the node shows is an error, never a silent 1-GPU run."""
    if requested < 1:
        raise SystemExit(f"bench.py: --gpus {requested}: need at least one GPU")
    if requested > visible:
        raise SystemExit(f"bench.py: --gpus {requested} requested but only {visible} CUDA device(s) are visible on this "
                         "node; refusing to report a smaller run under that label")


def main():
    args = parse_args()
    if args.impl != "reference" and "WORLD_SIZE" not in os.environ:
        check_gpus(args.gpus, torch.cuda.device_count() if torch.cuda.is_available() else 0)
        if args.gpus > 1:  # start the ranks ourselves: the line then reports n_gpus = the ranks that ran
            env = dict(os.environ)
            env.setdefault("NCCL_DEBUG", "INFO")  # the communicator's rank count is in the log (stderr)
            env.setdefault("NCCL_DEBUG_SUBSYS", "INIT")
            raise SystemExit(subprocess.call(launcher_command(args.gpus, sys.argv[1:]), env=env))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.impl == "reference":
        run_reference(args, rank)
        return
    if world != args.gpus:
        raise SystemExit(f"bench.py: --gpus {args.gpus} but the launcher started {world} rank(s); they must agree")
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback)")
    import paper_2606_31808_b200 as cd

    cd.lib()
    torch.cuda.set_device(local_rank)
    device = f"cuda:{local_rank}"
    dist = None
    if world > 1:
        import torch.distributed as dist_mod

        dist = dist_mod
        dist.init_process_group("nccl", device_id=torch.device(device))

    cfg = wl.CONFIGS[args.config]
    sz_logit, sz_mask = bytes_per_row_step(cfg)
    peak, peak_src = measured_peak()
    stream = torch.cuda.current_stream()

    # ---------------- c1-c3 beside the headline (rank 0; untimed for the others, who wait at the barrier)
    per_config = None
    if rank == 0 and not args.no_per_config and args.config == "c4" and args.gather_max == 0 and args.loop_mode == "auto":
        try:
            per_config = per_config_section(cd, device, peak, args.verbose)
        except Exception as ex:
            per_config = {"error": str(ex)[:300]}

    # weak scaling (default): every rank decodes its own batches of the table; strong scaling: ONE batch,
    # rank r takes the contiguous rows [r*B/N, (r+1)*B/N) (rows are independent, the automaton
    # is replicated, the concatenation of the ranks' results in rank order is the batch's -- no collective
    # on the data path)
    if args.scaling == "strong":
        lo, hi = wl.shard_rows(cfg.B, world, rank)
        aut, batches = build_inputs(cfg, device, args.batches, batch0=0, rows=(lo, hi))
        cfg = wl.scaled(cfg, B=hi - lo)
        rows_per_step_all_ranks = wl.CONFIGS[args.config].B
    else:
        aut, batches = build_inputs(cfg, device, args.batches, batch0=rank * args.batches)
        rows_per_step_all_ranks = cfg.B * world
    dfa = cd.compile_dfa(aut.V, aut.S, aut.start, aut.row_ptr, aut.tok, aut.next, aut.accepting, device=device)
    dfa.reserve(cfg.B)
    dfa.set_gather_max(args.gather_max)
    dfa.set_loop_mode({"auto": cd.LOOP_AUTO, "barrier": cd.LOOP_BARRIER, "per_step": cd.LOOP_PER_STEP}[args.loop_mode])
    out = None
    # One step = one cd_decode_loop over one resident batch.  The timed loops are enqueued back to back with
    # cd_decode_loop_async (arguments marshalled once per resident batch, every batch its own outputs); the
    # barrier() that closes the timed region synchronises the stream and checks the device-side status of
    # every loop (cd_loop_sync).
    loops = [cd.PreparedLoop(dfa, b, max_steps=cfg.max_steps) for b in batches]

    def one_step(i):
        nonlocal out
        out = loops[i % len(loops)].enqueue()

    def barrier():
        loops[0].sync()
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    # per-step active rows / distinct states / algorithmic bytes of every resident batch (untimed, through
    # the stepwise API); the event-timed replay of batch 0 gives the per-launch numbers of cd::step_kernel
    per_batch = []
    step_ms = []
    for b, logits in enumerate(batches):
        n_k, distinct_k, deg_k, t_k = replay_stepwise(cd, cfg, aut, dfa, logits, device, timed=(b == 0))
        per_batch.append(dict(n=n_k, distinct=distinct_k, deg=deg_k,
                              bytes=[n * sz_logit + d * sz_mask for n, d in zip(n_k, distinct_k)]))
        if b == 0:
            step_ms = t_k
    deg_k = per_batch[0]["deg"]
    deg_dev = torch.diff(torch.as_tensor(aut.row_ptr)).to(device)
    for i in range(args.warmup):
        one_step(i)
    barrier()
    sampler = ClockSampler(local_rank)
    sampler.start()
    launches0 = cd.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record(stream)
    for i in range(args.steps):
        one_step(args.warmup + i)
    e1.record(stream)
    barrier()
    launches = cd.launch_count() - launches0
    clocks = sampler.stop()
    ms = e0.elapsed_time(e1)
    tr_n, tr_ns = dfa.loop_trace()  # the last timed loop, step by step, from the persistent kernel's own trace
    if dist is not None:
        t = torch.tensor([ms], device=device)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms = float(t[0])
    value = rows_per_step_all_ranks * args.steps / (ms * 1e-3)
    timed = [(args.warmup + i) % len(batches) for i in range(args.steps)]
    row_steps_timed = sum(sum(per_batch[b]["n"]) for b in timed)
    row_steps = row_steps_timed / args.steps
    bytes_timed = sum(sum(per_batch[b]["bytes"]) for b in timed)

    # ---------------- roofline of the dominant kernel, live.
    # The whole loop is ONE launch of cd::loop_kernel, so "per launch" = per loop: algorithmic bytes of the
    # loop (every step's active rows x 512 KiB of logits + one 32 KiB mask row per distinct state) over the
    # CUDA-event duration of the timed region / K.  That duration also contains the loop's set-up kernel
    # and the host's hand-over between loops, so it is a lower bound of the kernel's own rate; the kernel's
    # device-side trace (cd_loop_trace) gives the per-step times of the last loop beside it.
    try:
        read_probe = cd.probe_read(batches[0][0], iters=10)
    except Exception:
        read_probe = None
    achieved = bytes_timed / (ms * 1e-3) / 1e9
    persistent = bool(tr_n) and tr_n == per_batch[timed[-1]]["n"]
    kname = ("cd::flow_kernel" if args.loop_mode == "auto" else "cd::loop_kernel") if persistent else "cd::step_kernel"
    tinfo = ncu_traffic(kname, cfg.name)
    roofline = {
        "bound": "hbm",
        "kernel": (kname + " (persistent: the whole decode loop in one launch; per row and step: fused mask read + masked "
                   "logsumexp/argmax + transition; " + ("every row advances on its own, no barrier)" if args.loop_mode == "auto"
                                                        else "grid barrier between steps)")) if persistent else
                  "cd::step_kernel (fused mask + masked logsumexp/argmax + CSR transition), one launch per decoding step",
        "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
        "peak_source": peak_src, "frac_of_nominal_8TBs": achieved / NOMINAL_HBM_GBS,
        "launches_timed": args.steps if persistent else int(row_steps and sum(len(per_batch[b]["n"]) for b in timed)),
        "bytes_per_launch_avg": bytes_timed / args.steps if persistent else bytes_timed / max(1, sum(len(per_batch[b]["n"]) for b in timed)),
        "us_per_launch_avg": 1e3 * ms / args.steps if persistent else 1e3 * ms / max(1, sum(len(per_batch[b]["n"]) for b in timed)),
        "duration_note": "CUDA events around the K timed cd_decode_loop_async calls (enqueued back to back, one cd_loop_sync after them) / K",
        "read_probe_gbs": read_probe, "frac_of_read_probe": (achieved / read_probe) if read_probe else None,
        "traffic": tinfo["bytes"] if tinfo else None,
        "traffic_source": (f"committed ncu --set full capture {tinfo['profile']} (one launch; not measured in this run)"
                           if tinfo else None),
    }
    if persistent:
        last = per_batch[timed[-1]]
        us = [t / 1e3 for t in tr_ns]
        kern_us = sum(us)
        gbs = [b / (max(t, 1) * 1e-9) / 1e9 for b, t in zip(last["bytes"], tr_ns)]
        roofline["device_trace"] = {
            "kernel_us_last_loop": kern_us, "kernel_gbs_last_loop": sum(last["bytes"]) / (kern_us * 1e-6) / 1e9,
            "kernel_frac_of_measured_peak": sum(last["bytes"]) / (kern_us * 1e-6) / 1e9 / peak,
            "kernel_share_of_loop_time": kern_us / (1e3 * ms / args.steps),
            "n_per_step": last["n"], "us_per_step": [round(u, 1) for u in us], "gbs_per_step": [round(g) for g in gbs],
            "best_step_gbs": max(gbs),
            "fixed_us_per_step_avg": sum(u - b / (READ_RATE_GBS * 1e3) for u, b in zip(us, last["bytes"])) / len(us),
        }
        if args.verbose and rank == 0:
            for k, (n, u, g) in enumerate(zip(last["n"], us, gbs)):
                print(f"  loop_kernel step {k:2d}: n={n:5d} distinct_states={last['distinct'][k]:5d} {u:8.1f} us {g:7.0f} GB/s",
                      file=sys.stderr)
    # cd::step_kernel (what cd_step launches: the stepwise API, the callback / host-buffer loops), per launch,
    # from the event-timed replay of batch 0
    if step_ms:
        sb = per_batch[0]["bytes"]
        tot_b, tot_ms = sum(sb), sum(step_ms)
        sk = ncu_traffic("cd::step_kernel", cfg.name)
        roofline["step_kernel"] = {
            "kernel": "cd::step_kernel (one launch per decoding step: cd_step)",
            "achieved": tot_b / (tot_ms * 1e-3) / 1e9, "frac": tot_b / (tot_ms * 1e-3) / 1e9 / peak,
            "frac_of_nominal_8TBs": tot_b / (tot_ms * 1e-3) / 1e9 / NOMINAL_HBM_GBS,
            "best_launch_gbs": max(bb / (mm * 1e-3) / 1e9 for bb, mm in zip(sb, step_ms)),
            "launches_timed": len(step_ms), "bytes_per_launch_avg": tot_b / len(step_ms),
            "us_per_launch_avg": 1e3 * tot_ms / len(step_ms),
            "traffic": sk["bytes"] if sk else None,
            "traffic_source": f"committed ncu --set full capture {sk['profile']} (the n = {per_batch[0]['n'][0]} launch)" if sk else None,
        }
        if args.verbose and rank == 0:
            for k, (mm, bb) in enumerate(zip(step_ms, sb)):
                print(f"  step_kernel step {k:2d}: n={per_batch[0]['n'][k]:5d} {1e3 * mm:8.1f} us {bb / (mm * 1e-3) / 1e9:7.0f} GB/s",
                      file=sys.stderr)

    # ---------------- density-adaptive step, reported beside the dense path:
    # the same loops with cd_set_gather_max(-1).  Its bytes are the bytes it touches (one 32-byte
    # sector + the 4-byte token id per allowed logit of a gathered row), never the dense count.
    adaptive = None
    if not args.no_adaptive and args.gather_max == 0:
        dfa.set_gather_max(-1)
        for i in range(args.warmup):
            one_step(i)
        barrier()
        a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a0.record(stream)
        for i in range(args.steps):
            one_step(args.warmup + i)
        a1.record(stream)
        barrier()
        ms_a = a0.elapsed_time(a1)
        if dist is not None:
            t = torch.tensor([ms_a], device=device)
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            ms_a = float(t[0])
        dfa.set_gather_max(0)
        auto_max = (sz_logit + sz_mask) // 232  # the library's automatic threshold (cd_api.cu gather_max_for)
        gathered = [dk for dk in deg_k]  # allowed logits per step of batch 0 (every row-step, if gathered)
        all_gathered = int(deg_dev.max()) <= auto_max
        adaptive = {
            "value": rows_per_step_all_ranks * args.steps / (ms_a * 1e-3), "unit": UNIT, "ms_per_step": ms_a / args.steps,
            "speedup_vs_dense": ms / ms_a, "gather_max": int(auto_max), "every_state_gathered": bool(all_gathered),
            "allowed_logits_per_loop_batch0": int(sum(gathered)),
            "touched_bytes_per_loop_batch0": int(sum(gathered)) * 36 if all_gathered else None,
            "note": "same outputs as the dense scan (parity-tested in gather modes); bytes = 32-byte sector + 4-byte "
                    "token id per allowed logit; DRAM moves 128-byte lines (profiles/r1d_gather_c4.md)",
        }
        if all_gathered:
            adaptive["touched_gbs"] = adaptive["touched_bytes_per_loop_batch0"] / (ms_a / args.steps * 1e-3) / 1e9

    # ---------------- sampled decoding: the same loops with cd_set_sampling(T = 1)
    sampling = None
    if not args.no_adaptive:
        dfa.set_sampling(1.0, seed=2026)
        for i in range(args.warmup):
            one_step(i)
        barrier()
        s0, s1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        s0.record(stream)
        for i in range(args.steps):
            one_step(args.warmup + i)
        s1.record(stream)
        barrier()
        ms_s = s0.elapsed_time(s1)
        rs_s = int(out["len"].sum())
        dfa.set_sampling(0.0)
        sampling = {"value": rows_per_step_all_ranks * args.steps / (ms_s * 1e-3), "unit": UNIT, "ms_per_step": ms_s / args.steps,
                    "slowdown_vs_greedy": ms_s / ms, "temperature": 1.0,
                    "row_steps_last_batch": rs_s,
                    "note": "Gumbel-max over the allowed set, counter-based noise per (row, step, token): one hash + two "
                            "fp32 logarithms per ALLOWED element; sampled rows take other paths through the automaton, so "
                            "row-steps per loop differ from the greedy run"}

    # ---------------- e2e: the same metric through the C ABI with HOST buffers
    e2e = None
    if not args.no_e2e:
        try:
            host = [torch.empty(x.shape, dtype=x.dtype, pin_memory=True) for x in batches[0]]
            for h, x in zip(host, batches[0]):
                h.copy_(x)
            torch.cuda.synchronize()
            out_h = None
            k_e2e = max(1, min(args.steps, 5))
            for i in range(1 + k_e2e):
                if i == 1:
                    barrier()
                    t0 = time.perf_counter()
                out_h = cd.decode_loop_host(dfa, host, max_steps=cfg.max_steps, out=out_h)
            barrier()
            dt = time.perf_counter() - t0
            if dist is not None:
                t = torch.tensor([dt], device=device)
                dist.all_reduce(t, op=dist.ReduceOp.MAX)
                dt = float(t[0])
            # the host loop copies only the rows still active at each step: one logits row per row-step
            steps_copied = int(out_h["len"].max())
            h2d = int(out_h["len"].sum()) * cfg.V * (2 if cfg.dtype == torch.bfloat16 else 4)
            d2h = cfg.B * (cfg.max_steps * 4 + 4 + 4 + 4 + 1) + 4 * steps_copied
            e2e = {"value": rows_per_step_all_ranks * k_e2e / dt, "unit": UNIT, "h2d_bytes_per_step": h2d,
                   "d2h_bytes_per_step": d2h, "steps": k_e2e, "ms_per_step": 1e3 * dt / k_e2e,
                   "h2d_gbs": h2d * k_e2e / dt / 1e9, "host_memory": "pinned"}
            got0 = cd.decode_loop(dfa, batches[0], max_steps=cfg.max_steps)
            assert torch.equal(out_h["tokens"], got0["tokens"].cpu()), "host-buffer loop disagrees with device loop"
            # the same with the density-adaptive step (cd_set_gather_max(-1)): when every state may be gathered the
            # step kernel pulls only the ALLOWED logits of the active rows over the link (a 32-byte sector each)
            if not args.no_adaptive and args.gather_max == 0:
                dfa.set_gather_max(-1)
                out_a = None
                for i in range(1 + k_e2e):
                    if i == 1:
                        barrier()
                        t0 = time.perf_counter()
                    out_a = cd.decode_loop_host(dfa, host, max_steps=cfg.max_steps, out=out_a)
                barrier()
                dta = time.perf_counter() - t0
                dfa.set_gather_max(0)
                assert torch.equal(out_a["tokens"], out_h["tokens"]), "adaptive host-buffer loop disagrees with the dense one"
                sectors = int(sum(deg_k)) * 32
                e2e["adaptive"] = {"value": rows_per_step_all_ranks * k_e2e / dta, "unit": UNIT, "ms_per_step": 1e3 * dta / k_e2e,
                                   "h2d_bytes_per_step": sectors, "h2d_gbs": sectors * k_e2e / dta / 1e9,
                                   "speedup_vs_dense": dt / dta,
                                   "note": "cd_set_gather_max(-1): same outputs; bytes = one 32-byte sector per allowed logit of "
                                           "an active row, read by the step kernel straight from the mapped host buffers "
                                           "(gathered only when every state has <= V / 32 transitions, else the dense path)"}
            del host
        except Exception as ex:  # e.g. not enough pinned host memory on this box
            e2e = {"value": None, "unit": UNIT, "error": str(ex)[:200]}

    # ---------------- CPU oracle timed beside it (rank 0, bounded sample, a baseline not a target)
    cpu = None
    if rank == 0 and not args.no_cpu_baseline:
        import oracle

        oracle.build()
        R = min(args.cpu_sample_rows, cfg.B)
        sub = [x[:R].cpu().contiguous() for x in batches[0]]
        t0 = time.perf_counter()
        reps = 0
        while True:
            res = oracle.decode_loop(aut, sub)
            reps += 1
            if time.perf_counter() - t0 > 12.0 or reps >= 400:
                break
        dt = time.perf_counter() - t0
        cpu = {"value": R * reps / dt, "unit": UNIT, "cores": 1, "host_cores": os.cpu_count(), "kind": "oracle",
               "sample": f"rows [0,{R}) of one {cfg.name} batch, all {cfg.max_steps} steps, {reps} passes, "
                         f"{int(res['n_active_hist'].sum())} row-steps per pass (D2H copy excluded)",
               "row_steps_per_s": int(res["n_active_hist"].sum()) * reps / dt}
        # parity spot check on the sample while we are here
        import numpy as np

        got = cd.decode_loop(dfa, batches[0], max_steps=cfg.max_steps)
        assert np.array_equal(got["tokens"][:R].cpu().numpy(), res["tokens"]), "bench parity check failed"

    head = None
    if rank == 0 and not args.no_head:
        try:
            head = head_section(cd, cfg, aut, dfa, device, args.head_H, max(3, min(args.steps, 10)), 3)
        except Exception as ex:
            head = {"error": str(ex)[:300]}

    dedup = None
    if rank == 0 and not args.no_dedup:
        try:
            dedup = dedup_section(cd, device, 20, 3)
        except Exception as ex:
            dedup = {"error": str(ex)[:300]}

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": args.scaling,
            "vs_baseline": None, "dtype": "f32", "logits_dtype": "bf16" if cfg.dtype == torch.bfloat16 else "f32",
            "data": "synthetic",
            "config": {
                "workload": f"{cfg.name}: {cfg.desc}; one step = cd_decode_loop over one batch of B={cfg.B} rows"
                            + (f"; {len(batches)} of the table's {cfg.n_batches} batches resident per GPU, rotated over the timed steps"
                               if getattr(cfg, "n_batches", 1) > 1 else f"; {len(batches)} seeded batches resident, rotated"),
                "B": cfg.B, "V": cfg.V, "max_steps": cfg.max_steps, "S": aut.S, "nnz": aut.nnz,
                "resident_batches": len(batches),
                "l2": f"inputs larger than L2: {cfg.max_steps * cfg.B * sz_logit / 2**30:.1f} GiB of logits per step, "
                      f"{len(batches)} batches rotated",
                "parallelism": (f"one batch of {rows_per_step_all_ranks} rows sharded over {world} GPU(s) ({cfg.B} rows each)"
                                if args.scaling == "strong" else f"every one of {world} GPU(s) decodes its own batches") +
                               ", automaton replicated, no collective",
                "loop_mode": args.loop_mode,
            },
            "row_steps_per_step": row_steps,
            "row_steps_per_s": row_steps_timed * world / (ms * 1e-3),  # rank 0's count x ranks
            "loop_gbs_per_gpu": row_steps_timed * sz_logit / (ms * 1e-3) / 1e9,
            "gpu_launches": launches,
            "clocks": clocks,
            "e2e": e2e,
            "roofline": roofline,
            "per_config": per_config,
            "adaptive": adaptive,
            "sampling": sampling,
            "cpu_baseline": cpu,
            "head": head,
            "dedup": dedup,
            "paper_context": "PAPER.md L17-18/L32: 390x lower cost, 3.8x lower latency than a proprietary API with a "
                             "quantized model on one 16 GB GPU; no per-step number is published (BASELINE.md)",
        }
        print(json.dumps(line), flush=True)
    dfa.close()
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
