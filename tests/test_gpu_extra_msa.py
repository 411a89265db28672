"""Extra-MSA stack (readings X.1-X.9) on the GPU vs oracle/extra_msa_ref.py, through the C ABI.
Tolerances of the bf16 path (north_star): max-abs 3e-2, mean-rel 1e-2 (R14) per sub-step and per block on unmasked
positions; every output finite."""
import numpy as np
import pytest

import paper_2111_06340_b200 as pf
import pf_synth as ps
from gpu_util import Margins, errors, valid_masks
from oracle import evoformer_sampled as osm
from oracle import extra_msa_ref as ex

pytestmark = pytest.mark.gpu

TOL_ABS, TOL_REL = 3e-2, 1e-2


def _run(blocks, e, z, sm, mm, block=None, substep=None, n_blocks=None):
    import torch
    h = pf.ExtraMsaStack(ps.pack_extra_blob(blocks), pf.make_extra_config(len(blocks)))
    ed, zd, smd, mmd = [torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in (e, z, sm, mm)]
    if substep is not None:
        h.forward_substep(ed, zd, smd, mmd, block or 0, substep)
    else:
        h.forward(ed, zd, smd, mmd, n_blocks if n_blocks is not None else len(blocks))
    torch.cuda.synchronize()
    n = h.last_launch_count()
    h.close()
    return ed.cpu().numpy(), zd.cpu().numpy(), n


def _oracle(blocks, e, z, sm, mm, block=None, substep=None):
    es, zs = [], []
    for b in range(e.shape[0]):
        if substep is not None:
            eo, zo = ex.substep(substep, e[b], z[b], sm[b], mm[b], blocks[block or 0])
        else:
            eo, zo = ex.extra_msa_stack(e[b], z[b], sm[b], mm[b], blocks)
        es.append(eo)
        zs.append(zo)
    return np.stack(es), np.stack(zs)


def _check(e, z, er, zr, sm, mm, what):
    vm, vz = valid_masks(sm, mm)
    em, rm = errors(e, er, vm)
    ez, rz = errors(z, zr, vz)
    print(f"{what}: e max-abs {em:.3e} mean-rel {rm:.3e}; z max-abs {ez:.3e} mean-rel {rz:.3e}")
    assert em <= TOL_ABS and ez <= TOL_ABS and rm <= TOL_REL and rz <= TOL_REL, (what, em, ez, rm, rz)


@pytest.fixture(scope="module")
def ragged():
    B, S, N = 2, 40, 72
    blocks = ps.make_extra_weights(131, 1, bf16_weights=True)
    e, z, sm, mm = ps.make_extra_inputs(132, B, S, N, lengths=[72, 51], msa_mask_frac_max=0.3)
    return blocks, e, z, sm, mm


@pytest.mark.parametrize("substep", range(1, 10))
def test_every_substep(ragged, substep):
    blocks, e, z, sm, mm = ragged
    eo, zo, _ = _run(blocks, e, z, sm, mm, block=0, substep=substep)
    er, zr = _oracle(blocks, e, z, sm, mm, block=0, substep=substep)
    _check(eo, zo, er, zr, sm, mm, f"extra substep {substep}")
    if substep <= 3:
        assert np.array_equal(zo, z)
    else:
        assert np.array_equal(eo, e)


def test_block_and_launch_count(ragged):
    blocks, e, z, sm, mm = ragged
    eo, zo, n = _run(blocks, e, z, sm, mm)
    er, zr = _oracle(blocks, e, z, sm, mm)
    _check(eo, zo, er, zr, sm, mm, "extra block")
    assert n >= 25


@pytest.mark.parametrize("B,S,N", [(1, 1, 9), (2, 600, 40), (1, 130, 129), (3, 17, 50)])
def test_runtime_shapes(B, S, N):
    """one binary, many shapes; N_seq = 600 takes two chunks of the outer-product contraction"""
    blocks = ps.make_extra_weights(133, 1, bf16_weights=True)
    lengths = ps.rng(B * 1000 + N, 7).integers(max(1, N // 2), N + 1, size=B)
    e, z, sm, mm = ps.make_extra_inputs(134, B, S, N, lengths=lengths, msa_mask_frac_max=0.4)
    eo, zo, _ = _run(blocks, e, z, sm, mm)
    er, zr = _oracle(blocks, e, z, sm, mm)
    _check(eo, zo, er, zr, sm, mm, f"extra B{B} S{S} N{N}")


def _substep_at(step, e, z, sm, mm, w, pos):
    if step == 1:
        return osm.msa_row_attention_at(e, z, sm, mm, w["row"], pos[0], pos[1], head_dim=8)
    if step == 2:
        return ex.msa_col_global_attention_at(e, sm, mm, w["col_global"], pos[0], pos[1], 8)
    if step == 3:
        return osm.transition_at(e[pos[0], pos[1]], w["msa_trans"])
    return osm.substep_at(step, e, z, sm, mm, w, pos, head_dim=32)


def test_paper_scale_extra_msa_sampled():
    """N_res 384 with 1,024 extra sequences (two outer-product chunks, 1,024 keys per column in the global attention), block 0,
    every sub-step teacher-forced, 32 sampled positions each against the one-position oracle functions."""
    import torch
    S, N = 1024, 384
    blocks = ps.make_extra_weights(135, 1, bf16_weights=True)
    g = torch.Generator(device="cuda").manual_seed(136)
    e = torch.randn((1, S, N, 64), device="cuda", generator=g)
    z = torch.randn((1, N, N, 128), device="cuda", generator=g)
    sm = np.ones((1, N), np.float32)
    mm = np.ones((1, S), np.float32)
    mm[0, 1 + ps.rng(137).choice(S - 1, size=200, replace=False)] = 0.0
    smd, mmd = torch.from_numpy(sm).cuda(), torch.from_numpy(mm).cuda()
    h = pf.ExtraMsaStack(ps.pack_extra_blob(blocks), pf.make_extra_config(1))
    for step in range(1, 10):
        e_in, z_in = e[0].cpu().numpy(), z[0].cpu().numpy()
        h.forward_substep(e, z, smd, mmd, 0, step)
        torch.cuda.synchronize()
        out = (e if step <= 3 else z)[0].cpu().numpy()
        assert np.isfinite(out).all()
        mg = Margins()
        for pos in ps.sample_positions(step, step, sm[0], mm[0], 32):
            mg.add(out[pos], _substep_at(step, e_in, z_in, sm[0], mm[0], blocks[0], pos))
        print(f"extra S=1024 N=384 substep {step}: max-abs {mg.max_abs:.3e} mean-rel {mg.mean_rel:.3e}")
        assert mg.max_abs <= TOL_ABS and mg.mean_rel <= TOL_REL, (step, mg.max_abs, mg.mean_rel)
    h.close()
