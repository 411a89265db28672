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
