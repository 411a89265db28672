"""Writes tests/golden/cfg1_block_samples.txt — sampled fp64 outputs of the oracle on BASELINE.json configs[0].

Calls only ``oracle/`` and ``pf_synth`` (never the CUDA path).  The paper prints no worked
numerical example of the Evoformer, so this fixture is a regression pin of the oracle itself: it makes any
later change to the oracle's arithmetic visible (and such a change must cite its justification in the commit).
Run from the repo root:  python tests/golden/make_golden.py
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import oracle  # noqa: E402
import pf_synth as ps  # noqa: E402

SEED, S, N = 1, 16, 32


def samples():
    w = ps.make_block_weights(SEED, 0)
    msa, pair, sm, mm = ps.make_inputs(SEED, 1, S, N)
    m, z = oracle.evoformer_block(msa[0], pair[0], sm[0], mm[0], w)
    g = ps.rng(SEED, 99)
    rows = []
    for _ in range(24):
        s, i, c = int(g.integers(S)), int(g.integers(N)), int(g.integers(256))
        rows.append(("m", s, i, c, m[s, i, c]))
    for _ in range(24):
        i, j, c = int(g.integers(N)), int(g.integers(N)), int(g.integers(128))
        rows.append(("z", i, j, c, z[i, j, c]))
    return rows


if __name__ == "__main__":
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "cfg1_block_samples.txt")
    with open(path, "w") as f:
        f.write("# oracle.evoformer_block on cfg1 (seed=1, S=16, N=32, AF2 dims, masks all 1); tensor i0 i1 c value(fp64)\n")
        f.write("# source: tests/golden/make_golden.py (oracle only); reading: SURVEY.md Appendix A, R0-R16\n")
        for t, a, b, c, v in samples():
            f.write(f"{t} {a} {b} {c} {float(v)!r}\n")
    print("wrote", path)
