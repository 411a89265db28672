"""bf16 CUDA path (tcgen05 tensor cores, fp32 accumulation, fp32 residual streams) vs the fp64 oracle, through the C ABI.

Tolerances (BASELINE.json north_star): max-abs 3e-2 and mean-rel 1e-2 per block output, mean-rel in the
ratio-of-means reading R14.  Weights are bf16-representable on both sides (R15).  Every sub-step is also gated on
its own (R16): the oracle is applied to the same fp32 input the GPU sub-step received (teacher forcing, R1).
"""
import numpy as np
import pytest

import paper_2111_06340_b200 as pf
import pf_synth as ps
from gpu_util import errors, run_cuda, run_oracle, valid_masks

pytestmark = pytest.mark.gpu

TOL_ABS, TOL_REL = 3e-2, 1e-2


@pytest.fixture(scope="module")
def ragged():
    """Several 128-row tiles with a ragged tail, masked residues and masked MSA rows, B > 1."""
    B, S, N = 2, 20, 72
    blocks = ps.make_weights(5, 1, bf16_weights=True)
    msa, pair, sm, mm = ps.make_inputs(6, B, S, N, lengths=[72, 51], msa_mask_frac_max=0.3)
    return blocks, msa, pair, sm, mm


def _check(m, z, mr, zr, sm, mm, what):
    vm, vz = valid_masks(sm, mm)
    em, rm = errors(m, mr, vm)
    ez, rz = errors(z, zr, vz)
    print(f"{what}: m max-abs {em:.3e} mean-rel {rm:.3e}; z max-abs {ez:.3e} mean-rel {rz:.3e}")
    assert em <= TOL_ABS and ez <= TOL_ABS, (what, em, ez)
    assert rm <= TOL_REL and rz <= TOL_REL, (what, rm, rz)


@pytest.mark.parametrize("substep", range(1, 10))
def test_every_substep(ragged, substep):
    blocks, msa, pair, sm, mm = ragged
    m, z = run_cuda(pf.PF_BF16, blocks, msa, pair, sm, mm, block=0, substep=substep)
    mr, zr = run_oracle(blocks, msa, pair, sm, mm, block=0, substep=substep)
    _check(m, z, mr, zr, sm, mm, f"substep {substep}")
    if substep <= 3:
        assert np.array_equal(z, pair)
    else:
        assert np.array_equal(m, msa)


def test_block(ragged):
    blocks, msa, pair, sm, mm = ragged
    m, z = run_cuda(pf.PF_BF16, blocks, msa, pair, sm, mm)
    mr, zr = run_oracle(blocks, msa, pair, sm, mm)
    _check(m, z, mr, zr, sm, mm, "block")


@pytest.mark.parametrize("B,S,N", [(1, 1, 9), (3, 17, 50), (1, 3, 129), (2, 130, 33),
                                   (2, 20, 64), (1, 40, 96), (2, 9, 48), (1, 64, 256)])
def test_runtime_shapes(B, S, N):
    """One binary, many shapes (H11): sizes that are not multiples of any tile, S=1, keys spanning two key tiles, and row
    tiles of every height (N = 64 / 96 / 48 / 256 -> 64 / 32 / 16 / 128 consecutive y per tile: the operand-swapped, TMA-staged
    and fallback store paths of the projection GEMM)."""
    blocks = ps.make_weights(8, 1, bf16_weights=True)
    lengths = ps.rng(B * 1000 + N, 7).integers(max(1, N // 2), N + 1, size=B)
    msa, pair, sm, mm = ps.make_inputs(9, B, S, N, lengths=lengths, msa_mask_frac_max=0.4)
    m, z = run_cuda(pf.PF_BF16, blocks, msa, pair, sm, mm)
    mr, zr = run_oracle(blocks, msa, pair, sm, mm)
    _check(m, z, mr, zr, sm, mm, f"B{B} S{S} N{N}")


def test_medium_protein_many_tiles():
    """A medium single protein with full masks plus one with a padded tail: N_res = 200 (two 128-query tiles, four 64-key
    tiles, row tiles of every geometry), N_seq = 96, one teacher-forced block checked element by element."""
    B, S, N = 2, 96, 200
    blocks = ps.make_weights(21, 1, bf16_weights=True)
    msa, pair, sm, mm = ps.make_inputs(22, B, S, N, lengths=[200, 131], msa_mask_frac_max=0.2)
    m, z = run_cuda(pf.PF_BF16, blocks, msa, pair, sm, mm)
    mr, zr = run_oracle(blocks, msa, pair, sm, mm)
    assert np.isfinite(m).all() and np.isfinite(z).all()
    _check(m, z, mr, zr, sm, mm, "medium protein")


@pytest.mark.parametrize("Np,Sp", [(140, 40), (192, 24), (128, 33)])
def test_masked_work_is_skipped_not_needed(Np, Sp):
    """Skipping of fully masked tiles / rows / key tiles (pf_flags.cu) must not change unmasked outputs: the same proteins
    embedded in a larger padded problem (bucket Np, N_seq Sp), with different garbage in the padding, give the same unmasked
    outputs up to the rounding of a different tile decomposition.  Run as ONE block so that later sub-steps see the stale
    workspace contents earlier sub-steps left at skipped positions (operands contracted over a masked index must be
    exact zeros there: this test failed before the kind-3 flags of pf_flags.cu)."""
    blocks = ps.make_weights(31, 1, bf16_weights=True)
    msa, pair, sm, mm = ps.make_inputs(32, 2, 24, 70, lengths=[70, 40], msa_mask_frac_max=0.3)
    m1, z1 = run_cuda(pf.PF_BF16, blocks, msa, pair, sm, mm)
    r = ps.rng(33, 1)
    msa2 = (3.0 * r.standard_normal((2, Sp, Np, 256))).astype(np.float32)
    pair2 = (3.0 * r.standard_normal((2, Np, Np, 128))).astype(np.float32)
    msa2[:, :24, :70] = msa
    pair2[:, :70, :70] = pair
    sm2 = np.zeros((2, Np), np.float32)
    sm2[:, :70] = sm
    mm2 = np.zeros((2, Sp), np.float32)
    mm2[:, :24] = mm
    m2, z2 = run_cuda(pf.PF_BF16, blocks, msa2, pair2, sm2, mm2)
    assert np.isfinite(m2).all() and np.isfinite(z2).all()
    vm, vz = valid_masks(sm, mm)
    em, rm = errors(m2[:, :24, :70], m1, vm)
    ez, rz = errors(z2[:, :70, :70], z1, vz)
    print(f"embedding: m max-abs {em:.3e} mean-rel {rm:.3e}; z max-abs {ez:.3e} mean-rel {rz:.3e}")
    assert em <= TOL_ABS and ez <= TOL_ABS and rm <= TOL_REL and rz <= TOL_REL
    mr, zr = run_oracle(blocks, msa, pair, sm, mm)
    _check(m2[:, :24, :70], z2[:, :70, :70], mr, zr, sm, mm, "embedded vs oracle")


def test_cfg2_full_size_sampled_proteins():
    """BASELINE.json configs[1] at full size in bench.py's launch configuration (B=64, N_seq=128, bucket 128, masks per
    R11), one teacher-forced block; the oracle recomputes two whole proteins of the batch (the two shortest, to bound
    CPU time) element by element, and every output of the batch must be finite."""
    B, S, N = 64, 128, 128
    blocks = ps.make_weights(7, 1, bf16_weights=True)
    lengths = ps.cfg2_lengths(100, B)
    msa, pair, sm, mm = ps.make_inputs(100, B, S, N, lengths=lengths, msa_mask_frac_max=0.3)
    m, z = run_cuda(pf.PF_BF16, blocks, msa, pair, sm, mm)
    assert np.isfinite(m).all() and np.isfinite(z).all()
    pick = np.argsort(lengths)[:2]
    for b in pick:
        sl = slice(int(b), int(b) + 1)
        mr, zr = run_oracle(blocks, msa[sl], pair[sl], sm[sl], mm[sl])
        _check(m[sl], z[sl], mr, zr, sm[sl], mm[sl], f"cfg2 protein {int(b)} (len {int(lengths[b])})")


@pytest.mark.parametrize("B", [1, 5, 11, 19])
def test_forward_host_pipelined_chunks_match_forward(B):
    """pf_evoformer_forward_host pipelines the batch in chunks of proteins over copy streams: every protein must come back
    exactly as from the device-resident call on the same batch (proteins are independent, so chunking changes nothing)."""
    import torch
    S, N = 12, 40
    blocks = ps.make_weights(41, 2, bf16_weights=True)
    lengths = ps.rng(42, B).integers(20, N + 1, size=B)
    msa, pair, sm, mm = ps.make_inputs(43, B, S, N, lengths=lengths, msa_mask_frac_max=0.3)
    valid_m, valid_z = valid_masks(sm, mm)
    m, z = run_cuda(pf.PF_BF16, blocks, msa, pair, sm, mm)
    h = pf.Evoformer(ps.pack_blob(blocks), pf.make_config(2, pf.PF_BF16))
    mh = torch.from_numpy(msa.copy()).pin_memory()
    zh = torch.from_numpy(pair.copy()).pin_memory()
    h.forward_host(mh, zh, torch.from_numpy(sm).pin_memory(), torch.from_numpy(mm).pin_memory(), 2)
    h.close()
    assert np.isfinite(mh.numpy()).all() and np.isfinite(zh.numpy()).all()
    assert np.array_equal(mh.numpy()[valid_m], m[valid_m]) and np.array_equal(zh.numpy()[valid_z], z[valid_z])


def test_chained_blocks_drift_reported():
    """Four chained blocks (no teacher forcing): the drift against the fp64 oracle is printed; the gate is loose
    (R1: per-block parity is the contract, chained drift is reported) — mean-rel 3e-2, every output finite."""
    B, S, N = 1, 24, 64
    blocks = ps.make_weights(51, 4, bf16_weights=True)
    msa, pair, sm, mm = ps.make_inputs(52, B, S, N, lengths=[57], msa_mask_frac_max=0.2)
    m, z = run_cuda(pf.PF_BF16, blocks, msa, pair, sm, mm)
    mr, zr = run_oracle(blocks, msa, pair, sm, mm)
    vm, vz = valid_masks(sm, mm)
    em, rm = errors(m, mr, vm)
    ez, rz = errors(z, zr, vz)
    print(f"4 chained blocks: m max-abs {em:.3e} mean-rel {rm:.3e}; z max-abs {ez:.3e} mean-rel {rz:.3e}")
    assert rm <= 3e-2 and rz <= 3e-2
