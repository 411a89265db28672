"""Seeded synthetic inputs and weights for the Evoformer trunk (shared by tests, bench and smoke).

This module holds NONE of the method's arithmetic: it only draws seeded random numbers, names the
parameters of one Evoformer block in the blob order of SURVEY.md Appendix B, and packs / unpacks
that blob.  Both the fp64 oracle (``oracle/``) and the CUDA path (``paper_2111_06340_b200``) are fed
from here so that they see bit-identical inputs; neither of them imports the other.

Readings used: R2 (mask shapes), R8 (init recipe), R10 (cfg5 length law),
R11 (cfg2 msa_mask law), R15 (weights are bf16-representable on the bf16 path).
Workload shapes stand in for the paper's data sets, which are not available:
PAPER.md:130-132 (small / medium / large sets), PAPER.md:113 (batches of similar-length proteins).
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np

# ----------------------------------------------------------------------------------------------
# dimensions (BASELINE.json north_star / configs[0]; SURVEY.md §8 header)
# ----------------------------------------------------------------------------------------------


@dataclass(frozen=True)
class Dims:
    c_m: int = 256
    c_z: int = 128
    heads_msa: int = 8
    heads_pair: int = 4
    head_dim: int = 32
    c_opm: int = 32
    c_tri: int = 128
    transition_n: int = 4


AF2 = Dims()


def _attn_spec(c, heads, with_pair_bias, c_bias_in):
    hd = c  # heads * head_dim == c
    spec = [("ln_g", (c,), "gamma"), ("ln_b", (c,), "beta")]
    if with_pair_bias == "row":
        spec += [("ln_z_g", (c_bias_in,), "gamma"), ("ln_z_b", (c_bias_in,), "beta")]
    if with_pair_bias:
        spec += [("w_bias", (c_bias_in, heads), "W")]
    spec += [("wq", (c, hd), "W"), ("wk", (c, hd), "W"), ("wv", (c, hd), "W"),
             ("wg", (c, hd), "W"), ("bg", (hd,), "bias"),
             ("wo", (hd, c), "W"), ("bo", (c,), "bias")]
    return spec


def block_spec(d: Dims = AF2):
    """Ordered list of (module, [(name, shape, kind)]) for one block — SURVEY.md Appendix B.

    kind: "W" (N(0,1)/sqrt(fan_in), bf16-rounded on the bf16 path), "bias" (0.1 N(0,1)),
    "gamma" (1 + 0.1 N(0,1)), "beta" (0.1 N(0,1))  — reading R8.
    """
    cm, cz, n = d.c_m, d.c_z, d.transition_n
    tri_mul = [("ln_in_g", (cz,), "gamma"), ("ln_in_b", (cz,), "beta"),
               ("w_ap", (cz, d.c_tri), "W"), ("b_ap", (d.c_tri,), "bias"),
               ("w_ag", (cz, d.c_tri), "W"), ("b_ag", (d.c_tri,), "bias"),
               ("w_bp", (cz, d.c_tri), "W"), ("b_bp", (d.c_tri,), "bias"),
               ("w_bg", (cz, d.c_tri), "W"), ("b_bg", (d.c_tri,), "bias"),
               ("w_g", (cz, cz), "W"), ("b_g", (cz,), "bias"),
               ("ln_out_g", (d.c_tri,), "gamma"), ("ln_out_b", (d.c_tri,), "beta"),
               ("w_z", (d.c_tri, cz), "W"), ("b_z", (cz,), "bias")]
    return [
        ("row", _attn_spec(cm, d.heads_msa, "row", cz)),
        ("col", _attn_spec(cm, d.heads_msa, None, 0)),
        ("msa_trans", [("ln_g", (cm,), "gamma"), ("ln_b", (cm,), "beta"),
                       ("w1", (cm, n * cm), "W"), ("b1", (n * cm,), "bias"),
                       ("w2", (n * cm, cm), "W"), ("b2", (cm,), "bias")]),
        ("opm", [("ln_g", (cm,), "gamma"), ("ln_b", (cm,), "beta"),
                 ("wa", (cm, d.c_opm), "W"), ("ba", (d.c_opm,), "bias"),
                 ("wb", (cm, d.c_opm), "W"), ("bb", (d.c_opm,), "bias"),
                 ("wout", (d.c_opm * d.c_opm, cz), "W"), ("bout", (cz,), "bias")]),
        ("tri_mul_out", list(tri_mul)),
        ("tri_mul_in", list(tri_mul)),
        ("tri_att_start", _attn_spec(cz, d.heads_pair, "self", cz)),
        ("tri_att_end", _attn_spec(cz, d.heads_pair, "self", cz)),
        ("pair_trans", [("ln_g", (cz,), "gamma"), ("ln_b", (cz,), "beta"),
                        ("w1", (cz, n * cz), "W"), ("b1", (n * cz,), "bias"),
                        ("w2", (n * cz, cz), "W"), ("b2", (cz,), "bias")]),
    ]


def block_floats(d: Dims = AF2) -> int:
    return sum(int(np.prod(shape)) for _, items in block_spec(d) for _, shape, _ in items)


# ----------------------------------------------------------------------------------------------
# random numbers: counter-based Philox, one stream per (seed, purpose)
# ----------------------------------------------------------------------------------------------

def rng(seed: int, stream: int = 0) -> np.random.Generator:
    return np.random.Generator(np.random.Philox(key=[int(seed) & 0xFFFFFFFFFFFFFFFF, int(stream)]))


def round_to_bf16(x: np.ndarray) -> np.ndarray:
    """Round fp32 to the nearest bf16-representable value (ties to even); returns fp32.

    Storage-format rounding of *parameters* (reading R15), not part of the method.
    """
    x = np.ascontiguousarray(x, dtype=np.float32)
    u = x.view(np.uint32).astype(np.uint64)
    lsb = (u >> 16) & 1
    u = (u + 0x7FFF + lsb) & 0xFFFF0000
    return u.astype(np.uint32).view(np.float32).reshape(x.shape)


def make_block_weights(seed: int, block: int, d: Dims = AF2, bf16_weights: bool = False):
    """dict[module][name] -> fp32 ndarray for one block (R8; R15 when bf16_weights)."""
    g = rng(seed, 1000 + block)
    out = {}
    for module, items in block_spec(d):
        mod = {}
        for name, shape, kind in items:
            r = g.standard_normal(shape, dtype=np.float32)
            if kind == "W":
                w = r / np.float32(np.sqrt(shape[0]))
                mod[name] = round_to_bf16(w) if bf16_weights else w.astype(np.float32)
            elif kind == "gamma":
                mod[name] = (1.0 + 0.1 * r).astype(np.float32)
            else:  # bias, beta
                mod[name] = (0.1 * r).astype(np.float32)
        out[module] = mod
    return out


def make_weights(seed: int, n_blocks: int, d: Dims = AF2, bf16_weights: bool = False):
    return [make_block_weights(seed, b, d, bf16_weights) for b in range(n_blocks)]


def pack_blob(blocks, d: Dims = AF2) -> np.ndarray:
    """Flatten a list of per-block weight dicts into the fp32 blob of Appendix B (row-major [in,out])."""
    parts = []
    for w in blocks:
        for module, items in block_spec(d):
            for name, shape, _ in items:
                a = np.asarray(w[module][name], dtype=np.float32)
                assert a.shape == tuple(shape), (module, name, a.shape, shape)
                parts.append(a.reshape(-1))
    return np.ascontiguousarray(np.concatenate(parts))


def unpack_blob(blob: np.ndarray, n_blocks: int, d: Dims = AF2):
    blob = np.asarray(blob, dtype=np.float32).reshape(-1)
    off, out = 0, []
    for _ in range(n_blocks):
        w = {}
        for module, items in block_spec(d):
            mod = {}
            for name, shape, _ in items:
                n = int(np.prod(shape))
                mod[name] = blob[off:off + n].reshape(shape).copy()
                off += n
            w[module] = mod
        out.append(w)
    assert off == blob.size
    return out


# ----------------------------------------------------------------------------------------------
# inputs
# ----------------------------------------------------------------------------------------------

def make_inputs(seed: int, B: int, S: int, N: int, d: Dims = AF2, lengths=None,
                msa_mask_frac_max: float = 0.0):
    """msa[B,S,N,c_m], pair[B,N,N,c_z] ~ N(0,1) everywhere, padding included (garbage, not zeros);
    seq_mask[b,i] = 1[i < lengths[b]] (R2); msa_mask per R11: per protein f ~ U[0, frac_max],
    floor(f*S) rows drawn without replacement from rows 1..S-1 are zeroed (row 0 always kept, R3).
    """
    g = rng(seed, 1)
    msa = g.standard_normal((B, S, N, d.c_m), dtype=np.float32)
    pair = g.standard_normal((B, N, N, d.c_z), dtype=np.float32)
    seq_mask = np.ones((B, N), dtype=np.float32)
    if lengths is not None:
        for b, L in enumerate(lengths):
            seq_mask[b, int(L):] = 0.0
    msa_mask = np.ones((B, S), dtype=np.float32)
    if msa_mask_frac_max > 0.0 and S > 1:
        gm = rng(seed, 2)
        for b in range(B):
            f = gm.uniform(0.0, msa_mask_frac_max)
            k = int(np.floor(f * S))
            if k > 0:
                rows = gm.choice(np.arange(1, S), size=min(k, S - 1), replace=False)
                msa_mask[b, rows] = 0.0
    return msa, pair, seq_mask, msa_mask


def cfg2_lengths(seed: int, B: int = 64, lo: int = 50, hi: int = 128) -> np.ndarray:
    """BASELINE.json configs[1]: lengths uniform in [lo, hi]."""
    return rng(seed, 3).integers(lo, hi + 1, size=B)


def cfg5_lengths(seed: int, n: int = 2000) -> np.ndarray:
    """BASELINE.json configs[4] with reading R10: log-normal(mu=ln 140, sigma=0.45), rounded, clipped to [50,300]."""
    x = rng(seed, 4).lognormal(mean=np.log(140.0), sigma=0.45, size=n)
    return np.clip(np.rint(x), 50, 300).astype(np.int64)


CFG5_BUCKETS = (64, 128, 192, 256, 320)


def gemm_flops_per_block(S: int, N: int, d: Dims = AF2) -> float:
    """Algorithmic GEMM FLOPs (2*MAC) of one block for one protein — SURVEY.md §8(d) formula F(S,N)."""
    cm, cz, co = d.c_m, d.c_z, d.c_opm
    return (36.0 * S * N * cm * cm + 4.0 * S * N * N * cm + 4.0 * N * S * S * cm
            + 4.0 * S * N * cm * co + 2.0 * S * N * N * co * co + 2.0 * N * N * co * co * cz
            + 60.0 * N * N * cz * cz + 12.0 * N ** 3 * cz
            + 2.0 * N * N * cz * d.heads_msa + 4.0 * N * N * cz * d.heads_pair)


def make_inputs_device(seed: int, B: int, S: int, N: int, device, d: Dims = AF2, lengths=None,
                       msa_mask_frac_max: float = 0.0):
    """make_inputs for batches too large to draw on the host in reasonable time (BASELINE.json configs[2..4] at full size):
    msa / pair ~ N(0,1) drawn by torch's seeded generator ON ``device`` (torch tensors, garbage in the padding as in
    make_inputs); the masks follow the same laws (R2, R11) and are returned as numpy arrays.  Whoever needs a protein's
    values on the host copies that slice back, so the oracle and the CUDA path still see identical bits."""
    import torch
    g = torch.Generator(device=device).manual_seed(int(seed))
    msa = torch.randn((B, S, N, d.c_m), device=device, generator=g, dtype=torch.float32)
    pair = torch.randn((B, N, N, d.c_z), device=device, generator=g, dtype=torch.float32)
    seq_mask = np.ones((B, N), dtype=np.float32)
    if lengths is not None:
        for b, L in enumerate(lengths):
            seq_mask[b, int(L):] = 0.0
    msa_mask = np.ones((B, S), dtype=np.float32)
    if msa_mask_frac_max > 0.0 and S > 1:
        gm = rng(seed, 2)
        for b in range(B):
            f = gm.uniform(0.0, msa_mask_frac_max)
            k = int(np.floor(f * S))
            if k > 0:
                rows = gm.choice(np.arange(1, S), size=min(k, S - 1), replace=False)
                msa_mask[b, rows] = 0.0
    return msa, pair, seq_mask, msa_mask


def sample_positions(seed: int, step: int, seq_mask_b, msa_mask_b, n: int):
    """n output positions of one protein for sub-step ``step`` at which a parity test compares the CUDA path with the
    sampled oracle: (s, i) with rho_s sigma_i = 1 for steps 1-3, (i, j) with sigma_i sigma_j = 1 for steps 4-9.  The corners
    of the unmasked region come first (first / last 128-row tile, first / last query and key tile), the rest is uniform."""
    res = np.flatnonzero(np.asarray(seq_mask_b) > 0.5)
    rows = np.flatnonzero(np.asarray(msa_mask_b) > 0.5)
    a, b = (rows, res) if step <= 3 else (res, res)
    pos = [(a[0], b[0]), (a[-1], b[-1]), (a[0], b[-1]), (a[-1], b[0]), (a[len(a) // 2], b[len(b) // 2])]
    g = rng(seed, 900 + step)
    while len(pos) < n:
        pos.append((a[int(g.integers(len(a)))], b[int(g.integers(len(b)))]))
    return [(int(p), int(q)) for p, q in pos[:n]]


# ----------------------------------------------------------------------------------------------
# input / recycling embedders (DESIGN.md §2b readings E.1-E.3)
# ----------------------------------------------------------------------------------------------

@dataclass(frozen=True)
class EmbedDims:
    c_m: int = 256
    c_z: int = 128
    tf_dim: int = 22          # target features: one break flag + 21 residue classes
    msa_dim: int = 49         # MSA features: 23 token classes + 2 deletion features + 23 profile entries + 1 deletion mean
    max_relpos: int = 32
    n_dist_bins: int = 15
    first_break: float = 3.25
    last_break: float = 20.75
    extra_dim: int = 25       # extra-MSA features: 23 token classes + 2 deletion features
    c_e: int = 64


EMBED = EmbedDims()


def embed_spec(d: EmbedDims = EMBED):
    """Ordered (name, shape, kind) of the embedder weights blob (row-major [in, out], as Appendix B)."""
    nrel = 2 * d.max_relpos + 1
    return [("w_a", (d.tf_dim, d.c_z), "W"), ("b_a", (d.c_z,), "bias"),
            ("w_b", (d.tf_dim, d.c_z), "W"), ("b_b", (d.c_z,), "bias"),
            ("w_rel", (nrel, d.c_z), "W"), ("b_rel", (d.c_z,), "bias"),
            ("w_m", (d.msa_dim, d.c_m), "W"), ("b_m", (d.c_m,), "bias"),
            ("w_t", (d.tf_dim, d.c_m), "W"), ("b_t", (d.c_m,), "bias"),
            ("ln_m_g", (d.c_m,), "gamma"), ("ln_m_b", (d.c_m,), "beta"),
            ("ln_z_g", (d.c_z,), "gamma"), ("ln_z_b", (d.c_z,), "beta"),
            ("w_d", (d.n_dist_bins, d.c_z), "W"), ("b_d", (d.c_z,), "bias"),
            ("w_e", (d.extra_dim, d.c_e), "W"), ("b_e", (d.c_e,), "bias")]


def make_embed_weights(seed: int, d: EmbedDims = EMBED):
    """R8 recipe; one-hot inputs select single rows, so W ~ N(0,1) (fan-in of a one-hot is 1) except the dense MSA features."""
    g = rng(seed, 2000)
    out = {}
    for name, shape, kind in embed_spec(d):
        r = g.standard_normal(shape, dtype=np.float32)
        if kind == "W":
            out[name] = (r / np.float32(np.sqrt(shape[0] if name == "w_m" else 1.0))).astype(np.float32)
        elif kind == "gamma":
            out[name] = (1.0 + 0.1 * r).astype(np.float32)
        else:
            out[name] = (0.1 * r).astype(np.float32)
    return out


def pack_embed_blob(w, d: EmbedDims = EMBED) -> np.ndarray:
    return np.ascontiguousarray(np.concatenate([np.asarray(w[n], dtype=np.float32).reshape(-1) for n, _, _ in embed_spec(d)]))


def make_features(seed: int, B: int, S: int, N: int, d: EmbedDims = EMBED):
    """Protein-shaped synthetic features (stand-ins for features.pkl, which needs the MSA stage):
    target_feat[B,N,22] one-hot residue classes, residue_index[B,N] = 0..N-1 with one chain gap, msa_feat[B,S,N,49]
    (one-hot token, deletion flags, a normalised profile), x_prev[B,N,3] a 3.8 Angstrom random walk (C-alpha-like trace,
    so pair distances cover all the distance bins)."""
    g = rng(seed, 2100)
    aa = g.integers(0, d.tf_dim - 1, size=(B, N))
    tf = np.zeros((B, N, d.tf_dim), np.float32)
    np.put_along_axis(tf, (aa + 1)[..., None], 1.0, axis=-1)
    ri = np.tile(np.arange(N, dtype=np.int32), (B, 1))
    for b in range(B):
        ri[b, N // 2:] += 20 * (b % 2)                      # a gap in the numbering of every other protein
    tok = g.integers(0, 23, size=(B, S, N))
    mf = np.zeros((B, S, N, d.msa_dim), np.float32)
    np.put_along_axis(mf[..., :23], tok[..., None], 1.0, axis=-1)
    mf[..., 23] = (g.uniform(size=(B, S, N)) < 0.1)
    mf[..., 24] = g.uniform(size=(B, S, N)).astype(np.float32) * mf[..., 23]
    prof = np.exp(g.standard_normal((B, 1, N, 23), dtype=np.float32))
    mf[..., 25:48] = prof / prof.sum(-1, keepdims=True)
    mf[..., 48] = g.uniform(size=(B, 1, N)).astype(np.float32) * 0.2
    step = g.standard_normal((B, N, 3), dtype=np.float32)
    step *= np.float32(3.8) / np.linalg.norm(step, axis=-1, keepdims=True)
    x = np.cumsum(step, axis=1).astype(np.float32)
    return tf, ri, mf, x


def make_extra_features(seed: int, B: int, S_e: int, N: int, d: EmbedDims = EMBED):
    """extra_msa_feat[B,S_e,N,25]: one-hot token + deletion flag + deletion value (stand-in for the unclustered sequences)."""
    g = rng(seed, 2200)
    tok = g.integers(0, 23, size=(B, S_e, N))
    xf = np.zeros((B, S_e, N, d.extra_dim), np.float32)
    np.put_along_axis(xf[..., :23], tok[..., None], 1.0, axis=-1)
    xf[..., 23] = (g.uniform(size=(B, S_e, N)) < 0.1)
    xf[..., 24] = g.uniform(size=(B, S_e, N)).astype(np.float32) * xf[..., 23]
    return xf


# ----------------------------------------------------------------------------------------------
# extra-MSA stack (DESIGN.md §2c readings X.1-X.9)
# ----------------------------------------------------------------------------------------------

@dataclass(frozen=True)
class ExtraDims:
    c_e: int = 64             # extra-MSA channels
    c_z: int = 128
    heads_msa: int = 8        # heads of dimension c_e / heads_msa = 8
    heads_pair: int = 4
    head_dim_pair: int = 32
    c_opm: int = 32
    c_tri: int = 128
    transition_n: int = 4

    @property
    def head_dim_msa(self):
        return self.c_e // self.heads_msa


EXTRA = ExtraDims()


def extra_block_spec(d: ExtraDims = EXTRA):
    """Ordered (module, [(name, shape, kind)]) of one extra-MSA block: as block_spec at c_m = c_e, with the column attention
    replaced by the global one (one shared key / value head of dimension head_dim_msa)."""
    main = Dims(c_m=d.c_e, c_z=d.c_z, heads_msa=d.heads_msa, heads_pair=d.heads_pair, head_dim=d.head_dim_pair,
                c_opm=d.c_opm, c_tri=d.c_tri, transition_n=d.transition_n)
    spec = block_spec(main)
    c, hd = d.c_e, d.head_dim_msa
    glob = [("ln_g", (c,), "gamma"), ("ln_b", (c,), "beta"), ("wq", (c, c), "W"), ("wk", (c, hd), "W"), ("wv", (c, hd), "W"),
            ("wg", (c, c), "W"), ("bg", (c,), "bias"), ("wo", (c, c), "W"), ("bo", (c,), "bias")]
    return [("col_global", glob) if mod == "col" else (mod, items) for mod, items in spec]


def extra_block_floats(d: ExtraDims = EXTRA) -> int:
    return sum(int(np.prod(shape)) for _, items in extra_block_spec(d) for _, shape, _ in items)


def make_extra_weights(seed: int, n_blocks: int, d: ExtraDims = EXTRA, bf16_weights: bool = False):
    out = []
    for blk in range(n_blocks):
        g = rng(seed, 3000 + blk)
        w = {}
        for module, items in extra_block_spec(d):
            mod = {}
            for name, shape, kind in items:
                r = g.standard_normal(shape, dtype=np.float32)
                if kind == "W":
                    v = r / np.float32(np.sqrt(shape[0]))
                    mod[name] = round_to_bf16(v) if bf16_weights else v.astype(np.float32)
                elif kind == "gamma":
                    mod[name] = (1.0 + 0.1 * r).astype(np.float32)
                else:
                    mod[name] = (0.1 * r).astype(np.float32)
            w[module] = mod
        out.append(w)
    return out


def pack_extra_blob(blocks, d: ExtraDims = EXTRA) -> np.ndarray:
    parts = []
    for w in blocks:
        for module, items in extra_block_spec(d):
            for name, shape, _ in items:
                a = np.asarray(w[module][name], dtype=np.float32)
                assert a.shape == tuple(shape), (module, name, a.shape, shape)
                parts.append(a.reshape(-1))
    return np.ascontiguousarray(np.concatenate(parts))


def make_extra_inputs(seed: int, B: int, S: int, N: int, d: ExtraDims = EXTRA, lengths=None, msa_mask_frac_max: float = 0.0):
    """e[B,S,N,c_e], z[B,N,N,c_z] ~ N(0,1) (garbage in the padding) and the masks of make_inputs."""
    main = Dims(c_m=d.c_e, c_z=d.c_z)
    return make_inputs(seed, B, S, N, main, lengths=lengths, msa_mask_frac_max=msa_mask_frac_max)


# ----------------------------------------------------------------------------------------------
# structure module + heads (DESIGN.md §2d readings M.0-M.6, H.1-H.5)
# ----------------------------------------------------------------------------------------------

@dataclass(frozen=True)
class StructDims:
    c_m: int = 256
    c_z: int = 128
    c_s: int = 384            # single representation
    heads: int = 12           # IPA heads
    c_ipa: int = 16           # scalar channels per head
    n_qp: int = 4             # query / key points per head
    n_pv: int = 8             # value points per head
    n_layers: int = 8         # layers, weights shared
    c_resnet: int = 128       # torsion-angle resnet width
    n_torsion: int = 7
    n_dist_bins: int = 64     # distogram head
    n_msa_classes: int = 23   # masked-MSA head
    n_lddt_bins: int = 50     # pLDDT head
    c_lddt: int = 128
    n_pae_bins: int = 64      # predicted-aligned-error head
    n_resolved: int = 37      # experimentally-resolved head (atom types)
    pos_scale: float = 10.0   # frame translations are in nanometres, positions in Angstrom

    @property
    def c_cat(self):          # width of the concatenated IPA outputs (M.2)
        return self.heads * (self.c_z + self.c_ipa + 4 * self.n_pv)


STRUCT = StructDims()


def struct_spec(d: StructDims = STRUCT):
    """Ordered (name, shape, kind) of the structure-module / heads blob (row-major [in, out], as Appendix B)."""
    cs, cz, cm, H, c, cr, cl = d.c_s, d.c_z, d.c_m, d.heads, d.c_ipa, d.c_resnet, d.c_lddt
    spec = [("w_single", (cm, cs), "W"), ("b_single", (cs,), "bias"),
            ("ln_s_g", (cs,), "gamma"), ("ln_s_b", (cs,), "beta"), ("ln_z_g", (cz,), "gamma"), ("ln_z_b", (cz,), "beta"),
            ("w_in", (cs, cs), "W"), ("b_in", (cs,), "bias"),
            ("w_q", (cs, H * c), "W"), ("w_k", (cs, H * c), "W"), ("w_v", (cs, H * c), "W"),
            ("w_qp", (cs, H * d.n_qp * 3), "W"), ("w_kp", (cs, H * d.n_qp * 3), "W"), ("w_vp", (cs, H * d.n_pv * 3), "W"),
            ("w_b", (cz, H), "W"), ("g_head", (H,), "bias"),
            ("w_out", (d.c_cat, cs), "W"), ("b_out", (cs,), "bias"),
            ("ln_ipa_g", (cs,), "gamma"), ("ln_ipa_b", (cs,), "beta")]
    for i in (1, 2, 3):
        spec += [(f"w_t{i}", (cs, cs), "W"), (f"b_t{i}", (cs,), "bias")]
    spec += [("ln_tr_g", (cs,), "gamma"), ("ln_tr_b", (cs,), "beta"),
             ("w_bb", (cs, 6), "W"), ("b_bb", (6,), "bias"),
             ("w_a1", (cs, cr), "W"), ("b_a1", (cr,), "bias"), ("w_a2", (cs, cr), "W"), ("b_a2", (cr,), "bias")]
    for r in (1, 2):
        spec += [(f"w_r{r}a", (cr, cr), "W"), (f"b_r{r}a", (cr,), "bias"), (f"w_r{r}b", (cr, cr), "W"), (f"b_r{r}b", (cr,), "bias")]
    spec += [("w_alpha", (cr, 2 * d.n_torsion), "W"), ("b_alpha", (2 * d.n_torsion,), "bias"),
             ("w_dg", (cz, d.n_dist_bins), "W"), ("b_dg", (d.n_dist_bins,), "bias"),
             ("w_mm", (cm, d.n_msa_classes), "W"), ("b_mm", (d.n_msa_classes,), "bias"),
             ("ln_l_g", (cs,), "gamma"), ("ln_l_b", (cs,), "beta"),
             ("w_l1", (cs, cl), "W"), ("b_l1", (cl,), "bias"), ("w_l2", (cl, cl), "W"), ("b_l2", (cl,), "bias"),
             ("w_l3", (cl, d.n_lddt_bins), "W"), ("b_l3", (d.n_lddt_bins,), "bias"),
             ("w_pae", (cz, d.n_pae_bins), "W"), ("b_pae", (d.n_pae_bins,), "bias"),
             ("w_er", (cs, d.n_resolved), "W"), ("b_er", (d.n_resolved,), "bias")]
    return spec


def struct_floats(d: StructDims = STRUCT) -> int:
    return sum(int(np.prod(shape)) for _, shape, _ in struct_spec(d))


def make_struct_weights(seed: int, d: StructDims = STRUCT):
    """R8 recipe (the structure module runs in fp32 on both sides: no bf16 rounding of its weights).  The backbone-update
    Linear is scaled by 0.3 so that eight layers of frame updates stay protein-sized (a walk of a few nanometres)."""
    g = rng(seed, 4000)
    out = {}
    for name, shape, kind in struct_spec(d):
        r = g.standard_normal(shape, dtype=np.float32)
        if kind == "W":
            out[name] = (r / np.float32(np.sqrt(shape[0])) * np.float32(0.3 if name == "w_bb" else 1.0)).astype(np.float32)
        elif kind == "gamma":
            out[name] = (1.0 + 0.1 * r).astype(np.float32)
        else:
            out[name] = (0.1 * r).astype(np.float32)
    return out


def pack_struct_blob(w, d: StructDims = STRUCT) -> np.ndarray:
    parts = []
    for name, shape, _ in struct_spec(d):
        a = np.asarray(w[name], dtype=np.float32)
        assert a.shape == tuple(shape), (name, a.shape, shape)
        parts.append(a.reshape(-1))
    return np.ascontiguousarray(np.concatenate(parts))
