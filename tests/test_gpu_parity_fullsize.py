"""bf16 CUDA path vs the fp64 oracle AT THE BENCHMARKED SIZES (BASELINE.json configs[1..4]), through the C ABI, in the launch
configuration bench.py times.  Whole-tensor fp64 evaluation is minutes per block there (SURVEY.md §8(c) "Feasibility"), so the
sampled-output oracle (oracle/evoformer_sampled.py, pinned to the full-tensor oracle in tests/test_oracle_sampled.py)
recomputes chosen output positions exactly: corners of the unmasked region (first / last row tile, first / last query and
key tile, the last outer-product k-block is part of every contraction) plus uniform draws.  Every sub-step is teacher-forced
(R1): the oracle sees the very fp32 tensors the GPU sub-step received.

Tolerances (north_star): max-abs 3e-2 and mean-rel 1e-2 (ratio of means, R14) per sub-step on unmasked positions.
"""
import numpy as np
import pytest

import paper_2111_06340_b200 as pf
import pf_synth as ps
from gpu_util import errors, run_oracle, sampled_substep_margins, valid_masks

pytestmark = pytest.mark.gpu

TOL_ABS, TOL_REL = 3e-2, 1e-2


def _gate(mg, what):
    print(f"{what}: max-abs {mg.max_abs:.3e} mean-rel {mg.mean_rel:.3e} over {mg.n} sampled outputs")
    assert mg.max_abs <= TOL_ABS and mg.mean_rel <= TOL_REL, (what, mg.max_abs, mg.mean_rel)


def _spread(lengths, k=4):
    """shortest, longest and k-2 proteins in between"""
    order = np.argsort(lengths, kind="stable")
    idx = sorted({int(order[0]), int(order[-1]), *[int(order[(len(order) * q) // (k - 1)]) for q in range(1, k - 1)]})
    return idx


def test_cfg2_four_proteins_four_blocks_teacher_forced():
    """configs[1] at full size (B=64, N_seq=128, bucket 128, masks R11): blocks 0..3 chained ON THE GPU; for every block the
    full fp64 oracle block is applied to the fp32 input the GPU block received, for four whole proteins (shortest, longest —
    no masked tile anywhere — and two in between), element by element."""
    import torch
    B, S, N, nb = 64, 128, 128, 4
    dev = torch.device("cuda:0")
    blocks = ps.make_weights(7, nb, bf16_weights=True)
    lengths = ps.cfg2_lengths(100, B)
    msa, pair, sm, mm = ps.make_inputs(100, B, S, N, lengths=lengths, msa_mask_frac_max=0.3)
    h = pf.Evoformer(ps.pack_blob(blocks), pf.make_config(nb, pf.PF_BF16))
    m, z = torch.from_numpy(msa).to(dev), torch.from_numpy(pair).to(dev)
    smd, mmd = torch.from_numpy(sm).to(dev), torch.from_numpy(mm).to(dev)
    pick = _spread(lengths, 4)
    assert max(lengths[b] for b in pick) == lengths.max() and min(lengths[b] for b in pick) == lengths.min()
    for blk in range(nb):
        ins = {b: (m[b].cpu().numpy(), z[b].cpu().numpy()) for b in pick}
        for step in range(1, 10):
            h.forward_substep(m, z, smd, mmd, blk, step)
        torch.cuda.synchronize()
        assert bool(torch.isfinite(m).all()) and bool(torch.isfinite(z).all())
        for b in pick:
            sl = slice(b, b + 1)
            mr, zr = run_oracle(blocks[blk:blk + 1], ins[b][0][None], ins[b][1][None], sm[sl], mm[sl])
            vm, vz = valid_masks(sm[sl], mm[sl])
            em, rm = errors(m[sl].cpu().numpy(), mr, vm)
            ez, rz = errors(z[sl].cpu().numpy(), zr, vz)
            print(f"cfg2 block {blk} protein {b} (len {int(lengths[b])}): m max-abs {em:.3e} mean-rel {rm:.3e}; "
                  f"z max-abs {ez:.3e} mean-rel {rz:.3e}")
            assert em <= TOL_ABS and ez <= TOL_ABS and rm <= TOL_REL and rz <= TOL_REL, (blk, b, em, ez, rm, rz)
    h.close()


def test_cfg2_forward_equals_substep_chain():
    """bench.py times pf_evoformer_forward; the teacher-forced tests drive pf_evoformer_forward_substep.  Both must be the
    same launch sequence: bit-identical outputs on a cfg2-shaped batch."""
    import torch
    B, S, N, nb = 8, 128, 128, 2
    dev = torch.device("cuda:0")
    blocks = ps.make_weights(7, nb, bf16_weights=True)
    lengths = ps.cfg2_lengths(101, B)
    msa, pair, sm, mm = ps.make_inputs(101, B, S, N, lengths=lengths, msa_mask_frac_max=0.3)
    h = pf.Evoformer(ps.pack_blob(blocks), pf.make_config(nb, pf.PF_BF16))
    smd, mmd = torch.from_numpy(sm).to(dev), torch.from_numpy(mm).to(dev)
    m1, z1 = torch.from_numpy(msa).to(dev), torch.from_numpy(pair).to(dev)
    h.forward(m1, z1, smd, mmd, nb)
    m2, z2 = torch.from_numpy(msa).to(dev), torch.from_numpy(pair).to(dev)
    for blk in range(nb):
        for step in range(1, 10):
            h.forward_substep(m2, z2, smd, mmd, blk, step)
    torch.cuda.synchronize()
    vm, vz = valid_masks(sm, mm)
    assert np.array_equal(m1.cpu().numpy()[vm], m2.cpu().numpy()[vm])
    assert np.array_equal(z1.cpu().numpy()[vz], z2.cpu().numpy()[vz])
    h.close()


@pytest.mark.parametrize("name,S,N", [("cfg3", 512, 384), ("cfg4", 512, 768)])
def test_single_protein_block0_every_substep(name, S, N):
    """configs[2] / configs[3]: one protein, full masks, N_seq 512 (8 outer-product k-blocks, 8 key tiles in column attention,
    3-6 query tiles per attention row, 6-12 k-blocks in the triangle einsum); block 0, every sub-step, 64 positions each."""
    import torch
    dev = torch.device("cuda:0")
    blocks = ps.make_weights(7, 1, bf16_weights=True)
    m, z, sm, mm = ps.make_inputs_device(300 + N, 1, S, N, dev)
    h = pf.Evoformer(ps.pack_blob(blocks), pf.make_config(1, pf.PF_BF16))
    for step in range(1, 10):
        mg = sampled_substep_margins(h, blocks, m, z, sm, mm, 0, step, [0], 64, seed=N)
        _gate(mg, f"{name} block 0 substep {step}")
    h.close()


def test_cfg3_late_blocks_teacher_forced():
    """configs[2], blocks 24 and 48 (indices 23, 47) of a 48-block trunk with distinct weights: the state is what the GPU's own
    chain produced (residual streams several times larger than N(0,1) by then); every sub-step of the block is teacher-forced
    against the sampled oracle; the chained state must stay finite."""
    import torch
    dev = torch.device("cuda:0")
    S, N, nb = 512, 384, 48
    blocks = ps.make_weights(7, nb, bf16_weights=True)
    m, z, sm, mm = ps.make_inputs_device(301, 1, S, N, dev)
    smd, mmd = torch.from_numpy(sm).to(dev), torch.from_numpy(mm).to(dev)
    h = pf.Evoformer(ps.pack_blob(blocks), pf.make_config(nb, pf.PF_BF16))
    done = 0
    for blk in (23, 47):
        for b in range(done, blk):
            for step in range(1, 10):
                h.forward_substep(m, z, smd, mmd, b, step)
        torch.cuda.synchronize()
        assert bool(torch.isfinite(m).all()) and bool(torch.isfinite(z).all())
        print(f"state before block {blk}: rms m {float(m.pow(2).mean().sqrt()):.2f}, rms z {float(z.pow(2).mean().sqrt()):.2f}")
        for step in range(1, 10):
            mg = sampled_substep_margins(h, blocks, m, z, sm, mm, blk, step, [0], 32, seed=blk)
            _gate(mg, f"cfg3 block {blk} substep {step}")
        done = blk + 1
    h.close()


def _cfg5_batches(S=512, cap=48, budget=16 << 30):
    """The batches bench.py's cfg5 sweep runs: 2,000 proteins (lengths R10) through pf_sched; the largest batch per bucket."""
    lengths = ps.cfg5_lengths(5, 2000)
    sched = pf.Scheduler(list(ps.CFG5_BUCKETS), budget, S)
    for i, L in enumerate(lengths):
        sched.add(i, int(L))
    best = {}
    for ids, lens, bucket in sched.batches(cap):
        if bucket not in best or len(ids) > len(best[bucket]):
            best[bucket] = lens
    sched.close()
    return best


@pytest.mark.parametrize("bucket", ps.CFG5_BUCKETS)
def test_cfg5_bucket_every_substep(bucket):
    """configs[4]: every length bucket at N_seq 512 with the batch size the scheduler gives bench.py (48 / 48 / 31 / 22 / 16
    proteins), seq_mask from the scheduled lengths, msa_mask R11; block 0, every sub-step, four proteins (shortest, longest,
    two in between) x 16 positions."""
    import torch
    dev = torch.device("cuda:0")
    S = 512
    lens = _cfg5_batches()[bucket]
    B = len(lens)
    blocks = ps.make_weights(7, 1, bf16_weights=True)
    m, z, sm, mm = ps.make_inputs_device(500 + bucket, B, S, bucket, dev, lengths=lens, msa_mask_frac_max=0.3)
    h = pf.Evoformer(ps.pack_blob(blocks), pf.make_config(1, pf.PF_BF16))
    pick = _spread(np.asarray(lens), 4)
    for step in range(1, 10):
        mg = sampled_substep_margins(h, blocks, m, z, sm, mm, 0, step, pick, 16, seed=bucket)
        _gate(mg, f"cfg5 bucket {bucket} (B={B}) substep {step}")
        assert bool(torch.isfinite(m if step <= 3 else z).all())
    h.close()


def test_handle_reuse_across_shrinking_shapes():
    """One handle, B = 48 then B = 44 at N_seq = N_res = 128 (the scheduler's tail batch of a bucket), then a smaller N_seq:
    the workspace layout depends on (B, S, N), so the second call lands on bytes the first one left in other formats.
    Padded lengths and a HOLE in seq_mask make partially masked tiles read what skipped tiles did not write.  Every output
    must be finite and two proteins per call must match the oracle."""
    import torch
    dev = torch.device("cuda:0")
    blocks = ps.make_weights(61, 1, bf16_weights=True)
    h = pf.Evoformer(ps.pack_blob(blocks), pf.make_config(1, pf.PF_BF16))
    for B, S, N in ((48, 128, 128), (44, 128, 128), (44, 60, 128), (5, 64, 120)):
        lengths = ps.cfg2_lengths(62 + B, B, lo=50, hi=N)
        msa, pair, sm, mm = ps.make_inputs(63 + B + S, B, S, N, lengths=lengths, msa_mask_frac_max=0.3)
        for b in range(B):
            sm[b, 10 + (b % 7)] = 0.0                       # a hole inside the protein
        m, z = torch.from_numpy(msa).to(dev), torch.from_numpy(pair).to(dev)
        h.forward(m, z, torch.from_numpy(sm).to(dev), torch.from_numpy(mm).to(dev), 1)
        torch.cuda.synchronize()
        mo, zo = m.cpu().numpy(), z.cpu().numpy()
        assert np.isfinite(mo).all() and np.isfinite(zo).all(), (B, S, N)
        for b in (int(np.argmin(lengths)), B - 1):
            sl = slice(b, b + 1)
            mr, zr = run_oracle(blocks, msa[sl], pair[sl], sm[sl], mm[sl])
            vm, vz = valid_masks(sm[sl], mm[sl])
            em, rm = errors(mo[sl], mr, vm)
            ez, rz = errors(zo[sl], zr, vz)
            print(f"reuse B={B} S={S} N={N} protein {b}: m {em:.3e}/{rm:.3e} z {ez:.3e}/{rz:.3e}")
            assert em <= TOL_ABS and ez <= TOL_ABS and rm <= TOL_REL and rz <= TOL_REL
    h.close()


def test_batches_beyond_one_launch_sequence_are_chunked():
    """B above the grid limit of one launch sequence (B * c_tri > 65535) is cut into chunks of proteins inside the library:
    the same proteins give the same results as in a small batch."""
    import torch
    dev = torch.device("cuda:0")
    B, S, N = 600, 2, 16
    blocks = ps.make_weights(65, 1, bf16_weights=True)
    lengths = ps.rng(66, 0).integers(8, N + 1, size=B)
    msa, pair, sm, mm = ps.make_inputs(67, B, S, N, lengths=lengths)
    h = pf.Evoformer(ps.pack_blob(blocks), pf.make_config(1, pf.PF_BF16))
    m, z = torch.from_numpy(msa).to(dev), torch.from_numpy(pair).to(dev)
    h.forward(m, z, torch.from_numpy(sm).to(dev), torch.from_numpy(mm).to(dev), 1)
    torch.cuda.synchronize()
    assert h.last_launch_count() > 2 * 25
    mo, zo = m.cpu().numpy(), z.cpu().numpy()
    assert np.isfinite(mo).all() and np.isfinite(zo).all()
    pick = [0, 299, 300, 599]
    m2 = torch.from_numpy(msa[pick]).to(dev)
    z2 = torch.from_numpy(pair[pick]).to(dev)
    h.forward(m2, z2, torch.from_numpy(sm[pick]).to(dev), torch.from_numpy(mm[pick]).to(dev), 1)
    torch.cuda.synchronize()
    vm, vz = valid_masks(sm[pick], mm[pick])
    assert np.array_equal(mo[pick][vm], m2.cpu().numpy()[vm]) and np.array_equal(zo[pick][vz], z2.cpu().numpy()[vz])
    mr, zr = run_oracle(blocks, msa[pick], pair[pick], sm[pick], mm[pick])
    em, rm = errors(mo[pick], mr, vm)
    ez, rz = errors(zo[pick], zr, vz)
    assert em <= TOL_ABS and ez <= TOL_ABS and rm <= TOL_REL and rz <= TOL_REL
    h.close()
