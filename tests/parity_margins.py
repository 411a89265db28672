#!/usr/bin/env python
"""Writes the parity-margin table (markdown on stdout) that profiles/rNN_parity_margins.md holds: for every shape the
-m gpu tests gate, per sub-step and per block, the bf16 CUDA path against the PLAIN fp64 oracle (the number the tolerances
apply to), the storage-rounding floor |quantised oracle - plain oracle| (R16: the oracle with 16-bit rounding at the
CUDA path's storage points, oracle/evoformer_sampled.py) and the remainder |GPU - quantised oracle|.

    python tests/parity_margins.py [--quick] > gpurun_out/parity_margins.md        (needs cuda:0)

Calls only the C ABI binding, pf_synth and oracle/; no value in it comes from anywhere else.
"""
import argparse
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(HERE))
sys.path.insert(0, HERE)

import paper_2111_06340_b200 as pf  # noqa: E402
import pf_synth as ps  # noqa: E402
from gpu_util import Margins, run_cuda, sampled_substep_margins, valid_masks  # noqa: E402
from oracle import evoformer_sampled as osm  # noqa: E402
import oracle  # noqa: E402

TOL_ABS, TOL_REL = 3e-2, 1e-2


def row(name, step, mg):
    ok = "ok" if (mg.max_abs <= TOL_ABS and mg.mean_rel <= TOL_REL) else "FAIL"
    print(f"| {name} | {step} | {mg.max_abs:.2e} | {mg.mean_rel:.2e} | {mg.floor:.2e} | {mg.resid:.2e} | {mg.n} | {ok} |", flush=True)


def small_block(name, dtype, seed, B, S, N, lengths, frac):
    """whole block, every position: GPU vs plain oracle vs quantised oracle (small shapes only)"""
    bf = dtype == pf.PF_BF16
    blocks = ps.make_weights(seed, 1, bf16_weights=bf)
    msa, pair, sm, mm = ps.make_inputs(seed + 1, B, S, N, lengths=lengths, msa_mask_frac_max=frac)
    m, z = run_cuda(dtype, blocks, msa, pair, sm, mm)
    vm, vz = valid_masks(sm, mm)
    gm, gz = Margins(), Margins()
    for b in range(B):
        mr, zr = oracle.evoformer_block(msa[b], pair[b], sm[b], mm[b], blocks[0])
        mq, zq = (osm.block_all(msa[b], pair[b], sm[b], mm[b], blocks[0], rnd=osm.Rounding(True)) if bf else (None, None))
        gm.add(m[b][vm[b]], mr[vm[b]], mq[vm[b]] if bf else None)
        gz.add(z[b][vz[b]], zr[vz[b]], zq[vz[b]] if bf else None)
    row(name, "block: m", gm)
    row(name, "block: z", gz)


def main():
    import torch
    ap = argparse.ArgumentParser()
    ap.add_argument("--quick", action="store_true", help="fewer sampled positions")
    args = ap.parse_args()
    npos = 8 if args.quick else 32
    dev = torch.device("cuda:0")
    print("# Parity margins: bf16 CUDA path vs fp64 oracle (tolerance max-abs 3e-2, mean-rel 1e-2 per sub-step / block)\n")
    print("Written by `python tests/parity_margins.py` on a B200.  `floor` = max-abs of (quantisation-aware oracle - plain oracle): "
          "what 16-bit storage costs by itself (R16); `gpu-quant` = max-abs of (GPU - quantisation-aware oracle): what is left "
          "for accumulation order, approximate exp2 / tanh and the model's simplifications.  fp32 path rows have no floor.\n")
    print("| shape | sub-step | max-abs vs plain | mean-rel vs plain | floor | gpu-quant | outputs compared | gate |")
    print("|---|---|---|---|---|---|---|---|")
    small_block("cfg1 fp32 (B1 S16 N32)", pf.PF_F32, 1, 1, 16, 32, None, 0.0)
    small_block("cfg1 shape, bf16 path", pf.PF_BF16, 1, 1, 16, 32, None, 0.0)
    small_block("ragged bf16 (B2 S20 N72)", pf.PF_BF16, 5, 2, 20, 72, [72, 51], 0.3)

    def sampled(name, seed, B, S, N, lengths, frac, pick, block=0, nb=1, pre_blocks=0):
        blocks = ps.make_weights(7, nb, bf16_weights=True)
        m, z, sm, mm = ps.make_inputs_device(seed, B, S, N, dev, lengths=lengths, msa_mask_frac_max=frac)
        h = pf.Evoformer(ps.pack_blob(blocks), pf.make_config(nb, pf.PF_BF16))
        if pre_blocks:
            h.forward(m, z, torch.from_numpy(sm).to(dev), torch.from_numpy(mm).to(dev), pre_blocks)
        for step in range(1, 10):
            mg = sampled_substep_margins(h, blocks, m, z, sm, mm, block, step, pick, npos, seed=N, quant=True)
            row(name, step, mg)
        h.close()
        del m, z
        torch.cuda.empty_cache()

    lengths = ps.cfg2_lengths(100, 64)
    order = np.argsort(lengths, kind="stable")
    sampled("cfg2 (B64 S128 N128), 4 proteins", 100, 64, 128, 128, lengths, 0.3,
            [int(order[0]), int(order[21]), int(order[42]), int(order[-1])])
    sampled("cfg3 (S512 N384) block 0", 684, 1, 512, 384, None, 0.0, [0])
    sampled("cfg3 block 47 after 47 GPU blocks", 301, 1, 512, 384, None, 0.0, [0], block=47, nb=48, pre_blocks=47)
    sampled("cfg4 (S512 N768) block 0", 1068, 1, 512, 768, None, 0.0, [0])
    if not args.quick:
        for bucket, B in ((64, 48), (128, 48), (192, 31), (256, 22), (320, 16)):
            lens = np.clip(ps.cfg5_lengths(5, 2000), 1, bucket)
            lens = np.sort(lens[(lens > bucket - 64) & (lens <= bucket)])[::-1][:B]
            o = np.argsort(lens, kind="stable")
            sampled(f"cfg5 bucket {bucket} (B{B} S512)", 500 + bucket, B, 512, bucket, lens, 0.3,
                    [int(o[0]), int(o[-1])])


if __name__ == "__main__":
    main()
