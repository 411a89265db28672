"""Input / recycling embedders and the recycled trunk (readings E.1-E.3) on the GPU vs oracle/embed_ref.py,
through the C ABI.  The embedders are fp32 elementwise work with reduction lengths <= 65: tolerance max-abs 1e-4 (the fp32
path's tolerance in north_star); the distance-bin decision is taken in fp32 on both sides and must agree exactly."""
import numpy as np
import pytest

import paper_2111_06340_b200 as pf
import pf_synth as ps
from gpu_util import errors, valid_masks
from oracle import embed_ref as er

pytestmark = pytest.mark.gpu


def _dev(*arrs):
    import torch
    return [torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in arrs]


@pytest.mark.parametrize("B,S,N", [(2, 5, 19), (1, 33, 70), (3, 2, 130)])
def test_embedder_first_cycle_and_recycle(B, S, N):
    import torch
    w = ps.make_embed_weights(91)
    tf, ri, mf, x = ps.make_features(92 + N, B, S, N)
    emb = pf.Embedder(ps.pack_embed_blob(w), pf.make_embed_config())
    tfd, rid, mfd, xd = _dev(tf, ri, mf, x)
    m = torch.full((B, S, N, 256), float("nan"), device="cuda")      # not read when has_prev = 0
    z = torch.full((B, N, N, 128), float("nan"), device="cuda")
    emb.forward(tfd, rid, mfd, xd, False, m, z)
    torch.cuda.synchronize()
    assert emb.last_launch_count() == 3
    for b in range(B):
        mr, zr = er.embed_cycle(tf[b], ri[b], mf[b], np.zeros((N, 256)), np.zeros((N, N, 128)), x[b], w)
        assert np.abs(m[b].cpu().numpy() - mr).max() < 1e-4 and np.abs(z[b].cpu().numpy() - zr).max() < 1e-4
    # second cycle, in place: the tensors now hold "the previous cycle's trunk output" (seeded values standing in for it)
    g = ps.rng(93)
    mp = (2.0 * g.standard_normal((B, S, N, 256))).astype(np.float32)
    zp = (3.0 * g.standard_normal((B, N, N, 128)) + 0.5).astype(np.float32)
    m, z = _dev(mp, zp)
    emb.forward(tfd, rid, mfd, xd, True, m, z)
    torch.cuda.synchronize()
    for b in range(B):
        mr, zr = er.embed_cycle(tf[b], ri[b], mf[b], mp[b, 0], zp[b], x[b], w)
        em, ez = np.abs(m[b].cpu().numpy() - mr).max(), np.abs(z[b].cpu().numpy() - zr).max()
        assert em < 1e-4 and ez < 1e-4, (b, em, ez)
    # no previous structure: NULL positions set no distance bin
    m, z = _dev(mp, zp)
    emb.forward(tfd, rid, mfd, None, True, m, z)
    torch.cuda.synchronize()
    mr, zr = er.embed_cycle(tf[0], ri[0], mf[0], mp[0, 0], zp[0], np.zeros((N, 3)), w)
    assert np.abs(z[0].cpu().numpy() - zr).max() < 1e-4
    emb.close()


def test_distance_bins_agree_exactly_near_the_edges():
    """Positions placed so that many pair distances sit within a few fp32 ulps of a bin edge: W_d rows are far apart (N(0,1)),
    so one flipped bin would show as an O(1) error."""
    import torch
    B, S, N = 1, 1, 96
    w = ps.make_embed_weights(94)
    tf, ri, mf, _ = ps.make_features(95, B, S, N)
    e = er.bin_edges(15, 3.25, 20.75)
    x = np.zeros((B, N, 3), np.float32)
    g = ps.rng(96)
    for i in range(1, N):                                   # residue i at distance edge_k (+- a few ulps) from residue 0
        d = np.float32(e[i % 15]) * np.float32(1.0 + (int(g.integers(-3, 4))) * 2.0 ** -23)
        u = g.standard_normal(3)
        x[0, i] = (u / np.linalg.norm(u)).astype(np.float32) * d
    emb = pf.Embedder(ps.pack_embed_blob(w), pf.make_embed_config())
    m = torch.zeros((B, S, N, 256), device="cuda")
    z = torch.zeros((B, N, N, 128), device="cuda")
    emb.forward(*_dev(tf, ri, mf, x), True, m, z)
    torch.cuda.synchronize()
    _, zr = er.embed_cycle(tf[0], ri[0], mf[0], np.zeros((N, 256)), np.zeros((N, N, 128)), x[0], w)
    assert np.abs(z[0].cpu().numpy() - zr).max() < 1e-4
    emb.close()


def test_recycled_trunk_matches_oracle():
    """E.3 with two cycles of a one-block trunk (bf16 path), two proteins with padding and masked MSA rows; tolerance of the
    bf16 path per block output (3e-2 / 1e-2) on unmasked positions — the second cycle starts from the first one's GPU output
    through LayerNorm, so this also checks that the in-place recycling reads the right rows."""
    import torch
    B, S, N, nb, cycles = 2, 12, 40, 1, 2
    w = ps.make_embed_weights(97)
    blocks = ps.make_weights(98, nb, bf16_weights=True)
    tf, ri, mf, x = ps.make_features(99, B, S, N)
    _, _, sm, mm = ps.make_inputs(99, B, S, N, lengths=[40, 27], msa_mask_frac_max=0.3)
    emb = pf.Embedder(ps.pack_embed_blob(w), pf.make_embed_config())
    evo = pf.Evoformer(ps.pack_blob(blocks), pf.make_config(nb, pf.PF_BF16))
    m = torch.empty((B, S, N, 256), device="cuda")
    z = torch.empty((B, N, N, 128), device="cuda")
    pf.forward_recycled(evo, emb, *_dev(tf, ri, mf, x), m, z, *_dev(sm, mm), nb, cycles)
    torch.cuda.synchronize()
    assert evo.last_launch_count() >= cycles * (3 + 25)
    mo, zo = m.cpu().numpy(), z.cpu().numpy()
    assert np.isfinite(mo).all() and np.isfinite(zo).all()
    for b in range(B):
        mr, zr = er.recycled_trunk(tf[b], ri[b], mf[b], x[b], sm[b], mm[b], w, blocks, cycles)
        vm, vz = valid_masks(sm[b:b + 1], mm[b:b + 1])
        em, rm = errors(mo[b:b + 1], mr[None], vm)
        ez, rz = errors(zo[b:b + 1], zr[None], vz)
        print(f"recycled trunk protein {b}: m {em:.3e}/{rm:.3e} z {ez:.3e}/{rz:.3e}")
        assert em <= 3e-2 and ez <= 3e-2 and rm <= 1e-2 and rz <= 1e-2
    emb.close()
    evo.close()


def test_recycled_trunk_with_extra_msa_stack_matches_oracle():
    """E.3 with the extra-MSA stack in every cycle: embedders -> e = Lin_e(extra features) -> one extra block -> one trunk
    block, two cycles."""
    import torch
    B, S, S_e, N, cycles = 2, 8, 70, 40, 2
    w = ps.make_embed_weights(141)
    blocks = ps.make_weights(142, 1, bf16_weights=True)
    xblocks = ps.make_extra_weights(143, 1, bf16_weights=True)
    tf, ri, mf, x = ps.make_features(144, B, S, N)
    xf = ps.make_extra_features(145, B, S_e, N)
    _, _, sm, mm = ps.make_inputs(146, B, S, N, lengths=[40, 31], msa_mask_frac_max=0.3)
    _, _, _, xm = ps.make_inputs(147, B, S_e, N, msa_mask_frac_max=0.3)
    emb = pf.Embedder(ps.pack_embed_blob(w), pf.make_embed_config())
    evo = pf.Evoformer(ps.pack_blob(blocks), pf.make_config(1, pf.PF_BF16))
    xst = pf.ExtraMsaStack(ps.pack_extra_blob(xblocks), pf.make_extra_config(1))
    m = torch.empty((B, S, N, 256), device="cuda")
    z = torch.empty((B, N, N, 128), device="cuda")
    e = torch.empty((B, S_e, N, 64), device="cuda")
    tfd, rid, mfd, xd, xfd, xmd, smd, mmd = _dev(tf, ri, mf, x, xf, xm, sm, mm)
    # E.4 alone first
    emb.forward_extra(xfd, e)
    torch.cuda.synchronize()
    assert np.abs(e[1].cpu().numpy() - er.extra_msa_embedder(xf[1], w)).max() < 1e-4
    pf.forward_recycled(evo, emb, tfd, rid, mfd, xd, m, z, smd, mmd, 1, cycles, extra=xst, extra_msa_feat=xfd, extra_msa=e,
                        extra_msa_mask=xmd, n_extra_blocks=1)
    torch.cuda.synchronize()
    mo, zo = m.cpu().numpy(), z.cpu().numpy()
    assert np.isfinite(mo).all() and np.isfinite(zo).all()
    for b in range(B):
        mr, zr = er.recycled_trunk(tf[b], ri[b], mf[b], x[b], sm[b], mm[b], w, blocks, cycles, extra=(xf[b], xm[b], xblocks, 8))
        vm, vz = valid_masks(sm[b:b + 1], mm[b:b + 1])
        em, rm = errors(mo[b:b + 1], mr[None], vm)
        ez, rz = errors(zo[b:b + 1], zr[None], vz)
        print(f"recycled trunk + extra stack protein {b}: m {em:.3e}/{rm:.3e} z {ez:.3e}/{rz:.3e}")
        assert em <= 3e-2 and ez <= 3e-2 and rm <= 1e-2 and rz <= 1e-2
    for o in (emb, evo, xst):
        o.close()
