"""Writes tests/golden/c1_tokens.txt — calls ONLY oracle/ (and the seeded input generator).

Regression fixture, not a paper value: the paper prints no worked numeric example (all of
its numbers are inside figure images).  Run:  python tests/golden/make_golden.py
"""
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import m2r2_synth as S  # noqa: E402
from oracle import Oracle  # noqa: E402


def main():
    cfg = S.config_c1()
    W = S.gen_weights(cfg)
    o = Oracle(cfg, W)
    toks = [o.prefill(S.gen_prompt(cfg, 32))]
    for _ in range(31):
        toks.append(o.decode_step()[0])
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "c1_tokens.txt")
    with open(path, "w") as fh:
        fh.write("# C1 (BASELINE.json configs[0]) plain greedy decode: prompt 32 -> 32 tokens.\n")
        fh.write("# Written by tests/golden/make_golden.py from oracle/ only.\n")
        fh.write(" ".join(str(t) for t in toks) + "\n")
    print(path, toks)


if __name__ == "__main__":
    main()
