"""Writes tests/golden/*.txt.  Calls ONLY oracle/ and the seeded generators in
workloads/ (never the CUDA path).  Re-run by hand after a justified oracle
change:  python tests/golden/make_golden.py

The paper prints no numeric example of a decoding step,
so these fixtures are not "the paper's values": they are the oracle's results
on BASELINE.json configs[0] (tiny boolean) and on a reduced configs[3] recipe,
frozen so that (a) an accidental change of the oracle's arithmetic or of the
generators shows up as a diff and (b) the GPU tests have a stored, oracle-made
expectation that does not depend on the oracle being buildable on the box.
"""
import os
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))

import oracle  # noqa: E402
import workloads as wl  # noqa: E402


def dump(path, header, res):
    B, K = res["tokens"].shape
    with open(path, "w") as f:
        f.write(header)
        f.write("# row len done final_state sum_logprob(%.17g) tokens...\n")
        for r in range(B):
            toks = " ".join(str(int(t)) for t in res["tokens"][r])
            f.write(f"{r} {int(res['len'][r])} {int(res['done'][r])} {int(res['final_state'][r])} "
                    f"{float(res['sum_logprob'][r]):.17g} {toks}\n")
        f.write("# n_active_hist " + " ".join(str(int(x)) for x in res["n_active_hist"]) + "\n")


def cases():
    c0 = wl.CONFIGS["c0"]
    yield "c0_decode.txt", c0, "# BASELINE.json configs[0] (tiny boolean), CPU-generated fp32 logits, oracle O4\n"
    c3 = wl.scaled(wl.CONFIGS["c3"], V=4096, B=48, S=64, max_steps=10)
    yield "c3_small_decode.txt", c3, "# reduced configs[3] recipe: V=4096 B=48 S=64 10 steps bf16, oracle O4\n"


def main():
    for name, cfg, header in cases():
        aut = wl.build_automaton(cfg)
        logits = wl.build_step_logits(cfg, aut, device="cpu")
        res = oracle.decode_loop(aut, logits)
        dump(os.path.join(HERE, name), header, res)
        print("wrote", name)


if __name__ == "__main__":
    main()
