"""Helpers for the -m gpu parity tests: run the CUDA path through the C ABI, run the oracle, compare (R3, R14)."""
import numpy as np

import oracle
import paper_2111_06340_b200 as pf
import pf_synth as ps


def run_cuda(dtype, blocks, msa, pair, seq_mask, msa_mask, n_blocks=None, block=None, substep=None, handle=None):
    """Returns (m, z) as numpy fp32 after forward (or one substep) on cuda:0."""
    import torch
    dev = torch.device("cuda:0")
    own = handle is None
    if own:
        blob = ps.pack_blob(blocks)
        handle = pf.Evoformer(blob, pf.make_config(len(blocks), dtype))
    m = torch.from_numpy(np.ascontiguousarray(msa, dtype=np.float32)).to(dev)
    z = torch.from_numpy(np.ascontiguousarray(pair, dtype=np.float32)).to(dev)
    sm = torch.from_numpy(np.ascontiguousarray(seq_mask, dtype=np.float32)).to(dev)
    mm = torch.from_numpy(np.ascontiguousarray(msa_mask, dtype=np.float32)).to(dev)
    if substep is not None:
        handle.forward_substep(m, z, sm, mm, block or 0, substep)
    else:
        handle.forward(m, z, sm, mm, n_blocks if n_blocks is not None else len(blocks))
    torch.cuda.synchronize()
    out = m.cpu().numpy(), z.cpu().numpy()
    if own:
        handle.close()
    return out


def run_oracle(blocks, msa, pair, seq_mask, msa_mask, block=None, substep=None):
    ms, zs = [], []
    for b in range(msa.shape[0]):
        if substep is not None:
            m, z = oracle.substep(substep, msa[b], pair[b], seq_mask[b], msa_mask[b], blocks[block or 0])
        else:
            m, z = oracle.evoformer_trunk(msa[b], pair[b], seq_mask[b], msa_mask[b], blocks)
        ms.append(m)
        zs.append(z)
    return np.stack(ms), np.stack(zs)


def errors(got, ref, valid):
    """max-abs and ratio-of-means relative error (R14) over unmasked positions; got must be finite everywhere (R3)."""
    assert np.isfinite(got).all(), "non-finite output"
    g = got[valid].astype(np.float64)
    r = ref[valid]
    diff = np.abs(g - r)
    return float(diff.max()), float(diff.mean() / np.abs(r).mean())


def valid_masks(seq_mask, msa_mask):
    vm = (msa_mask[:, :, None] * seq_mask[:, None, :]) > 0          # [B,S,N]
    vz = (seq_mask[:, :, None] * seq_mask[:, None, :]) > 0          # [B,N,N]
    return vm, vz


# ------------------------------------------------------------------------------------------------
# sampled parity at the benchmarked sizes (oracle/evoformer_sampled.py): the CUDA path runs ONE sub-step on device-resident
# tensors (teacher forcing: the oracle sees the very fp32 input the GPU sub-step received), chosen proteins are copied back
# and compared at sampled positions
# ------------------------------------------------------------------------------------------------
class Margins:
    """max-abs and ratio-of-means relative error (R14) accumulated over sampled positions, against the plain oracle;
    with quant=True also the storage-rounding floor |quantised - plain| and the remainder |gpu - quantised| (R16)."""

    def __init__(self):
        self.max_abs = 0.0
        self.sum_diff = 0.0
        self.sum_ref = 0.0
        self.n = 0
        self.floor = 0.0
        self.resid = 0.0

    def add(self, got, ref, quant=None):
        got = np.asarray(got, dtype=np.float64)
        assert np.isfinite(got).all(), "non-finite output"
        d = np.abs(got - ref)
        self.max_abs = max(self.max_abs, float(d.max()))
        self.sum_diff += float(d.sum())
        self.sum_ref += float(np.abs(ref).sum())
        self.n += got.size
        if quant is not None:
            self.floor = max(self.floor, float(np.abs(quant - ref).max()))
            self.resid = max(self.resid, float(np.abs(got - quant).max()))

    @property
    def mean_rel(self):
        return self.sum_diff / max(self.sum_ref, 1e-300)


def sampled_substep_margins(handle, blocks, m_dev, z_dev, sm, mm, block, step, proteins, n_pos, seed=0, quant=False):
    """Runs sub-step ``step`` of block ``block`` IN PLACE on the device tensors and returns the Margins of the updated
    stream at ``n_pos`` sampled positions of each protein in ``proteins``.  sm / mm: numpy masks of the whole batch."""
    import torch
    from oracle import evoformer_sampled as osm
    dev = m_dev.device
    smd, mmd = torch.from_numpy(sm).to(dev), torch.from_numpy(mm).to(dev)
    ins = {int(b): (m_dev[b].cpu().numpy(), z_dev[b].cpu().numpy()) for b in proteins}
    handle.forward_substep(m_dev, z_dev, smd, mmd, block, step)
    torch.cuda.synchronize()
    mg = Margins()
    rnd = osm.Rounding(True) if quant else None
    for b in proteins:
        b = int(b)
        m_in, z_in = ins[b]
        out = (m_dev if step <= 3 else z_dev)[b].cpu().numpy()
        other_in, other_out = (z_in, z_dev[b]) if step <= 3 else (m_in, m_dev[b])
        assert np.array_equal(other_out.cpu().numpy(), other_in), "the stream a sub-step does not own changed"
        for pos in ps.sample_positions(seed + 17 * b, step, sm[b], mm[b], n_pos):
            ref = osm.substep_at(step, m_in, z_in, sm[b], mm[b], blocks[block], pos)
            q = osm.substep_at(step, m_in, z_in, sm[b], mm[b], blocks[block], pos, rnd=rnd) if quant else None
            mg.add(out[pos], ref, q)
    return mg
