"""Pins of oracle/embed_ref.py (input / recycling embedders, recycled trunk; DESIGN.md §2b readings E.1-E.3)."""
import math

import numpy as np
import pytest

import pf_synth as ps
from oracle import embed_ref as er
from oracle import evoformer_ref as ref


@pytest.fixture(scope="module")
def case():
    S, N = 4, 11
    w = ps.make_embed_weights(81)
    tf, ri, mf, x = ps.make_features(82, 2, S, N)
    return w, tf[1], ri[1], mf[1], x[1]


def test_one_hot_linears_are_row_gathers(case):
    """a one-hot times W is the selected row: z_ij = W_a[aa_i] + b_a + W_b[aa_j] + b_b + W_rel[rel_ij] + b_rel."""
    w, tf, ri, mf, x = case
    m, z = er.input_embedder(tf, ri, mf, w)
    aa = tf.argmax(-1)
    N = len(aa)
    for i in (0, 3, N - 1):
        for j in (0, 5, N - 1):
            rel = min(max(int(ri[i]) - int(ri[j]), -32), 32) + 32
            ref_z = (w["w_a"][aa[i]].astype(np.float64) + w["b_a"] + w["w_b"][aa[j]] + w["b_b"] + w["w_rel"][rel] + w["b_rel"])
            assert np.abs(z[i, j] - ref_z).max() < 1e-12
    # i and j are not interchangeable (W_a != W_b, rel index antisymmetric): a transposed z fails this
    assert np.abs(z - np.transpose(z, (1, 0, 2))).max() > 0.1
    s, i = 2, 7
    ref_m = mf[s, i].astype(np.float64) @ w["w_m"].astype(np.float64) + w["b_m"] + w["w_t"][aa[i]] + w["b_t"]
    assert np.abs(m[s, i] - ref_m).max() < 1e-12


def test_relpos_index_properties():
    r = np.array([0, 1, 2, 50, 51, 120])
    idx = er.relpos_index(r, 32)
    assert np.array_equal(idx + idx.T, np.full_like(idx, 64)) and (np.diag(idx) == 32).all()
    assert idx[0, 1] == 31 and idx[1, 0] == 33 and idx[0, 3] == 0 and idx[5, 0] == 64


def test_distance_bins_match_searchsorted_and_edges():
    """K lower edges 3.25 .. 20.75 step 1.25; d in (e_k, e_{k+1}) -> bin k; below 3.25 no bin; beyond 20.75 the last bin."""
    e = er.bin_edges(15, 3.25, 20.75)
    assert np.allclose(np.diff(e), 1.25) and e[0] == 3.25 and e[-1] == 20.75
    g = ps.rng(83)
    x = (g.uniform(-12, 12, size=(40, 3))).astype(np.float32)
    oh = er.distance_one_hot(x, 15, 3.25, 20.75)
    d = np.sqrt(((x[:, None].astype(np.float64) - x[None].astype(np.float64)) ** 2).sum(-1))
    k = np.searchsorted(e, d, side="left") - 1            # library routine: index of the last edge below d
    far = np.abs(d[..., None] - e).min(-1) > 1e-4         # away from the edges the fp32 decision equals the fp64 one
    assert far.mean() > 0.99
    for i, j in zip(*np.nonzero(far)):
        if k[i, j] < 0:
            assert oh[i, j].sum() == 0
        else:
            assert oh[i, j].sum() == 1 and oh[i, j, k[i, j]] == 1
    assert oh[np.arange(40), np.arange(40)].sum() == 0      # d = 0: all-zero one-hot
    assert oh.sum(-1).max() == 1


def test_recycling_embedder_brute_force(case):
    w, tf, ri, mf, x = case
    g = ps.rng(84)
    N, S = len(ri), mf.shape[0]
    m, z = er.input_embedder(tf, ri, mf, w)
    m0p, zp = g.standard_normal((N, 256)), g.standard_normal((N, N, 128))
    m2, z2 = er.recycling_embedder(m, z, m0p, zp, x, w)
    edges = [3.25 + 1.25 * k for k in range(15)]

    def ln(v, gam, bet):
        mu = sum(v) / len(v)
        var = sum((t - mu) ** 2 for t in v) / len(v)
        return [(t - mu) / math.sqrt(var + 1e-5) * float(a) + float(b) for t, a, b in zip(v, gam, bet)]

    for i, j in ((0, 0), (1, 9), (10, 2)):
        d = math.sqrt(sum((float(x[i, c]) - float(x[j, c])) ** 2 for c in range(3)))
        k = max([q for q in range(15) if d > edges[q]], default=-1)
        lnz = ln([float(t) for t in zp[i, j]], w["ln_z_g"], w["ln_z_b"])
        for c in (0, 77, 127):
            exp = float(z[i, j, c]) + lnz[c] + float(w["b_d"][c]) + (float(w["w_d"][k, c]) if k >= 0 else 0.0)
            assert abs(z2[i, j, c] - exp) < 1e-10
    lnm = ln([float(t) for t in m0p[4]], w["ln_m_g"], w["ln_m_b"])
    assert abs(m2[0, 4, 9] - (m[0, 4, 9] + lnm[9])) < 1e-10
    assert np.array_equal(m2[1:], m[1:])                    # only the first MSA row is recycled


def test_first_cycle_closed_form(case):
    """Previous representations and positions all zero: LN(0) = beta, no distance bin -> z += ln_z_b + b_d, m_0 += ln_m_b."""
    w, tf, ri, mf, x = case
    N = len(ri)
    m, z = er.input_embedder(tf, ri, mf, w)
    m2, z2 = er.recycling_embedder(m, z, np.zeros((N, 256)), np.zeros((N, N, 128)), np.zeros((N, 3)), w)
    assert np.abs(z2 - (z + w["ln_z_b"].astype(np.float64) + w["b_d"])).max() < 1e-12
    assert np.abs(m2[0] - (m[0] + w["ln_m_b"].astype(np.float64))).max() < 1e-12


def test_recycled_trunk_is_the_cycle_loop(tiny_dims):
    """E.3 with n_cycles = 2 equals embed -> trunk -> embed(with the first cycle's m_0, z) -> trunk written out by hand; with
    identity blocks (all output weights zero) the second cycle's input is LN of the first cycle's embedding."""
    d = ps.EmbedDims(c_m=tiny_dims.c_m, c_z=tiny_dims.c_z)
    w = ps.make_embed_weights(85, d)
    tf, ri, mf, x = ps.make_features(86, 1, 3, 6, d)
    blocks = ps.make_weights(87, 1, tiny_dims)
    sig, rho = np.ones(6), np.ones(3)
    hd = tiny_dims.head_dim
    got_m, got_z = er.recycled_trunk(tf[0], ri[0], mf[0], x[0], sig, rho, w, blocks, 2, head_dim=hd)
    m, z = er.embed_cycle(tf[0], ri[0], mf[0], np.zeros((6, d.c_m)), np.zeros((6, 6, d.c_z)), x[0], w)
    m, z = ref.evoformer_trunk(m, z, sig, rho, blocks, hd)
    m, z = er.embed_cycle(tf[0], ri[0], mf[0], m[0], z, x[0], w)
    m, z = ref.evoformer_trunk(m, z, sig, rho, blocks, hd)
    assert np.abs(got_m - m).max() < 1e-12 and np.abs(got_z - z).max() < 1e-12
    one = er.recycled_trunk(tf[0], ri[0], mf[0], x[0], sig, rho, w, blocks, 1, head_dim=hd)
    assert np.abs(one[1] - got_z).max() > 1e-3              # the second cycle changes the result


def test_recycled_trunk_with_extra_msa_stack(tiny_dims):
    """E.3 with the extra-MSA stack: per cycle embed -> e = Lin_e(features) -> extra stack (only z leaves it) -> trunk, written
    out by hand; the stack must change the result."""
    from oracle import extra_msa_ref as xr
    d = ps.EmbedDims(c_m=tiny_dims.c_m, c_z=tiny_dims.c_z, c_e=4)
    xd = ps.ExtraDims(c_e=4, c_z=tiny_dims.c_z, heads_msa=2, heads_pair=tiny_dims.heads_pair, head_dim_pair=tiny_dims.head_dim,
                      c_opm=tiny_dims.c_opm, c_tri=tiny_dims.c_tri, transition_n=tiny_dims.transition_n)
    w = ps.make_embed_weights(88, d)
    tf, ri, mf, x = ps.make_features(89, 1, 3, 6, d)
    xf = ps.make_extra_features(90, 1, 5, 6, d)
    blocks = ps.make_weights(91, 1, tiny_dims)
    xblocks = ps.make_extra_weights(92, 1, xd)
    sig, rho, xrho = np.ones(6), np.ones(3), np.array([1.0, 1, 0, 1, 1])
    hd = tiny_dims.head_dim
    got = er.recycled_trunk(tf[0], ri[0], mf[0], x[0], sig, rho, w, blocks, 2, head_dim=hd,
                            extra=(xf[0], xrho, xblocks, xd.head_dim_msa))
    m0p, zp = np.zeros((6, d.c_m)), np.zeros((6, 6, d.c_z))
    for _ in range(2):
        m, z = er.embed_cycle(tf[0], ri[0], mf[0], m0p, zp, x[0], w)
        e = xf[0].astype(np.float64) @ w["w_e"].astype(np.float64) + w["b_e"]
        _, z = xr.extra_msa_stack(e, z, sig, xrho, xblocks, xd.head_dim_msa, hd)
        m, z = ref.evoformer_trunk(m, z, sig, rho, blocks, hd)
        m0p, zp = m[0], z
    assert np.abs(got[0] - m).max() < 1e-12 and np.abs(got[1] - z).max() < 1e-12
    plain = er.recycled_trunk(tf[0], ri[0], mf[0], x[0], sig, rho, w, blocks, 2, head_dim=hd)
    assert np.abs(plain[1] - got[1]).max() > 1e-3
