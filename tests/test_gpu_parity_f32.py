"""fp32 CUDA path vs the fp64 oracle, element by element, through the C ABI (BASELINE.json configs[0]).

Tolerance (north_star): max-abs 1e-4 per block output for the fp32 path.
"""
import numpy as np
import pytest

import paper_2111_06340_b200 as pf
import pf_synth as ps
from gpu_util import errors, run_cuda, run_oracle, valid_masks

pytestmark = pytest.mark.gpu

TOL_F32 = 1e-4


@pytest.fixture(scope="module")
def cfg1():
    blocks = ps.make_weights(1, 1)
    msa, pair, sm, mm = ps.make_inputs(1, 1, 16, 32)
    return blocks, msa, pair, sm, mm


@pytest.mark.parametrize("substep", range(1, 10))
def test_cfg1_every_substep(cfg1, substep):
    blocks, msa, pair, sm, mm = cfg1
    m, z = run_cuda(pf.PF_F32, blocks, msa, pair, sm, mm, block=0, substep=substep)
    mr, zr = run_oracle(blocks, msa, pair, sm, mm, block=0, substep=substep)
    vm, vz = valid_masks(sm, mm)
    em, _ = errors(m, mr, vm)
    ez, _ = errors(z, zr, vz)
    assert em <= TOL_F32 and ez <= TOL_F32, (substep, em, ez)
    # the stream a sub-step does not own is bit-identical to its input
    if substep <= 3:
        assert np.array_equal(z, pair)
    else:
        assert np.array_equal(m, msa)


def test_cfg1_block(cfg1):
    blocks, msa, pair, sm, mm = cfg1
    m, z = run_cuda(pf.PF_F32, blocks, msa, pair, sm, mm)
    mr, zr = run_oracle(blocks, msa, pair, sm, mm)
    vm, vz = valid_masks(sm, mm)
    em, rm = errors(m, mr, vm)
    ez, rz = errors(z, zr, vz)
    print(f"cfg1 block fp32: m max-abs {em:.3e} rel {rm:.3e}; z max-abs {ez:.3e} rel {rz:.3e}")
    assert em <= TOL_F32 and ez <= TOL_F32


@pytest.mark.parametrize("B,S,N", [(2, 5, 13), (1, 1, 9), (3, 17, 50), (1, 3, 77)])
def test_ragged_shapes_with_masks(B, S, N):
    """Runtime shapes with one binary (H11): odd sizes, tails that are not tile multiples, masked residues and rows."""
    blocks = ps.make_weights(3, 2)
    lengths = ps.rng(B * 1000 + N, 7).integers(max(1, N // 2), N + 1, size=B)
    msa, pair, sm, mm = ps.make_inputs(4, B, S, N, lengths=lengths, msa_mask_frac_max=0.5)
    m, z = run_cuda(pf.PF_F32, blocks, msa, pair, sm, mm)
    mr, zr = run_oracle(blocks, msa, pair, sm, mm)
    vm, vz = valid_masks(sm, mm)
    em, _ = errors(m, mr, vm)
    ez, _ = errors(z, zr, vz)
    assert em <= 3 * TOL_F32 and ez <= 3 * TOL_F32, (em, ez)   # two chained blocks


def test_forward_host_matches_forward(cfg1):
    import torch
    blocks, msa, pair, sm, mm = cfg1
    m, z = run_cuda(pf.PF_F32, blocks, msa, pair, sm, mm)
    h = pf.Evoformer(ps.pack_blob(blocks), pf.make_config(1, pf.PF_F32))
    mh = torch.from_numpy(msa.copy()).pin_memory()
    zh = torch.from_numpy(pair.copy()).pin_memory()
    h.forward_host(mh, zh, torch.from_numpy(sm), torch.from_numpy(mm), 1)
    assert np.array_equal(mh.numpy(), m) and np.array_equal(zh.numpy(), z)
    assert h.last_launch_count() > 0
    h.close()


def test_error_paths(cfg1):
    import torch
    blocks, msa, pair, sm, mm = cfg1
    blob = ps.pack_blob(blocks)
    with pytest.raises(pf.PfError):
        pf.Evoformer(blob[:-1], pf.make_config(1, pf.PF_F32))
    with pytest.raises(pf.PfError):
        pf.Evoformer(blob, pf.make_config(1, pf.PF_F32, head_dim=16, heads_msa=16, heads_pair=8))
    h = pf.Evoformer(blob, pf.make_config(1, pf.PF_F32))
    t = torch.zeros(1, device="cuda")
    with pytest.raises(pf.PfError):
        h.forward(torch.zeros(1, 2, 2, 256, device="cuda"), torch.zeros(1, 2, 2, 128, device="cuda"), t, t, 2)
    h.close()
