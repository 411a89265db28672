"""Thin ctypes binding over the C ABI of include/pf_evoformer.h (argument marshalling only).

Every step of the Evoformer trunk runs in the CUDA kernels of ``csrc/``; this module only loads
``libpf_evoformer.so`` (built in-tree by ``python -m paper_2111_06340_b200.build``), converts arguments to
pointers and sizes, and raises on non-OK status.  There is no CPU fallback: if the library is missing or a
call fails, an exception is raised.  The fp64 oracle under ``oracle/`` is never imported from here.
"""
from __future__ import annotations

import ctypes
import os
from ctypes import POINTER, Structure, byref, c_char_p, c_float, c_int, c_longlong, c_size_t, c_void_p

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libpf_evoformer.so")

PF_OK = 0
PF_F32, PF_BF16 = 0, 1
STATUS_NAMES = {0: "PF_OK", 1: "PF_ERR_INVALID_ARG", 2: "PF_ERR_SHAPE", 3: "PF_ERR_ALLOC", 4: "PF_ERR_CUDA",
                5: "PF_ERR_ARCH", 6: "PF_ERR_UNIMPLEMENTED"}

EXPORTED_SYMBOLS = (
    "pf_evoformer_block_floats", "pf_evoformer_create", "pf_evoformer_forward", "pf_evoformer_forward_substep",
    "pf_evoformer_forward_host", "pf_evoformer_workspace_bytes", "pf_evoformer_last_launch_count",
    "pf_evoformer_set_profiling", "pf_evoformer_profile_kinds", "pf_evoformer_profile_name",
    "pf_evoformer_get_profile", "pf_evoformer_profile_records", "pf_evoformer_get_profile_record", "pf_evoformer_destroy", "pf_last_error", "pf_sched_create", "pf_sched_add", "pf_sched_next_batch",
    "pf_sched_bytes_per_protein", "pf_sched_cost", "pf_sched_partition", "pf_sched_destroy",
    "pf_embedder_floats", "pf_embedder_create", "pf_embedder_forward", "pf_embedder_forward_extra",
    "pf_embedder_last_launch_count", "pf_embedder_destroy",
    "pf_evoformer_forward_recycled",
    "pf_extra_msa_block_floats", "pf_extra_msa_create", "pf_extra_msa_forward", "pf_extra_msa_forward_substep",
    "pf_extra_msa_last_launch_count", "pf_extra_msa_set_profiling", "pf_extra_msa_get_profile", "pf_extra_msa_destroy",
    "pf_structure_floats", "pf_structure_create", "pf_structure_forward", "pf_heads_forward",
    "pf_structure_last_launch_count", "pf_structure_destroy", "pf_fold_forward", "pf_plddt_forward_static",
)


class PfConfig(Structure):
    _fields_ = [("c_m", c_int), ("c_z", c_int), ("heads_msa", c_int), ("heads_pair", c_int), ("head_dim", c_int),
                ("c_opm", c_int), ("c_tri", c_int), ("transition_n", c_int), ("n_blocks_max", c_int),
                ("dtype", c_int)]


class PfEmbedConfig(Structure):
    _fields_ = [("c_m", c_int), ("c_z", c_int), ("tf_dim", c_int), ("msa_dim", c_int), ("max_relpos", c_int),
                ("n_dist_bins", c_int), ("first_break", c_float), ("last_break", c_float), ("extra_dim", c_int),
                ("c_e", c_int)]


class PfExtraConfig(Structure):
    _fields_ = [("c_e", c_int), ("c_z", c_int), ("heads_msa", c_int), ("heads_pair", c_int), ("head_dim_pair", c_int),
                ("c_opm", c_int), ("c_tri", c_int), ("transition_n", c_int), ("n_blocks_max", c_int)]


class PfStructConfig(Structure):
    _fields_ = [("c_m", c_int), ("c_z", c_int), ("c_s", c_int), ("heads", c_int), ("c_ipa", c_int), ("n_qp", c_int),
                ("n_pv", c_int), ("n_layers", c_int), ("c_resnet", c_int), ("n_torsion", c_int), ("n_dist_bins", c_int),
                ("n_msa_classes", c_int), ("n_lddt_bins", c_int), ("c_lddt", c_int), ("n_pae_bins", c_int), ("n_resolved", c_int),
                ("pos_scale", c_float)]


class PfError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__(f"{STATUS_NAMES.get(status, status)}: {msg}")
        self.status = status


_lib = None


def lib() -> ctypes.CDLL:
    """Load the shared library (once).  Raises if it has not been built — never falls back."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} not built; run `python -m paper_2111_06340_b200.build`")
        L = ctypes.CDLL(LIB_PATH)
        L.pf_evoformer_block_floats.restype = c_size_t
        L.pf_evoformer_block_floats.argtypes = [POINTER(PfConfig)]
        L.pf_evoformer_create.restype = c_int
        L.pf_evoformer_create.argtypes = [POINTER(c_void_p), c_void_p, c_size_t, POINTER(PfConfig)]
        fwd = [c_void_p, c_void_p, c_void_p, c_void_p, c_void_p, c_int, c_int, c_int]
        L.pf_evoformer_forward.restype = c_int
        L.pf_evoformer_forward.argtypes = fwd + [c_int, c_void_p]
        L.pf_evoformer_forward_substep.restype = c_int
        L.pf_evoformer_forward_substep.argtypes = fwd + [c_int, c_int, c_void_p]
        L.pf_evoformer_forward_host.restype = c_int
        L.pf_evoformer_forward_host.argtypes = fwd + [c_int, c_void_p]
        L.pf_evoformer_workspace_bytes.restype = c_size_t
        L.pf_evoformer_workspace_bytes.argtypes = [c_void_p, c_int, c_int, c_int]
        L.pf_evoformer_last_launch_count.restype = c_longlong
        L.pf_evoformer_last_launch_count.argtypes = [c_void_p]
        L.pf_evoformer_set_profiling.restype = c_int
        L.pf_evoformer_set_profiling.argtypes = [c_void_p, c_int]
        L.pf_evoformer_profile_kinds.restype = c_int
        L.pf_evoformer_profile_kinds.argtypes = []
        L.pf_evoformer_profile_name.restype = c_char_p
        L.pf_evoformer_profile_name.argtypes = [c_int]
        L.pf_evoformer_get_profile.restype = c_int
        L.pf_evoformer_get_profile.argtypes = [c_void_p, c_int, POINTER(c_longlong), POINTER(ctypes.c_double),
                                               POINTER(ctypes.c_double), POINTER(ctypes.c_double)]
        L.pf_evoformer_profile_records.restype = c_longlong
        L.pf_evoformer_profile_records.argtypes = [c_void_p]
        L.pf_evoformer_get_profile_record.restype = c_int
        L.pf_evoformer_get_profile_record.argtypes = [c_void_p, c_longlong, POINTER(c_int), POINTER(ctypes.c_double),
                                                      POINTER(ctypes.c_double), POINTER(ctypes.c_double)]
        L.pf_evoformer_destroy.restype = None
        L.pf_evoformer_destroy.argtypes = [c_void_p]
        L.pf_last_error.restype = c_char_p
        L.pf_sched_create.restype = c_int
        L.pf_sched_create.argtypes = [POINTER(c_void_p), POINTER(c_int), c_int, c_size_t, c_int]
        L.pf_sched_add.restype = c_int
        L.pf_sched_add.argtypes = [c_void_p, c_int, c_int]
        L.pf_sched_next_batch.restype = c_int
        L.pf_sched_next_batch.argtypes = [c_void_p, POINTER(c_int), POINTER(c_int), c_int, POINTER(c_int)]
        L.pf_sched_bytes_per_protein.restype = c_size_t
        L.pf_sched_bytes_per_protein.argtypes = [c_int, c_int]
        L.pf_sched_cost.restype = ctypes.c_double
        L.pf_sched_cost.argtypes = [c_int, c_int]
        L.pf_sched_partition.restype = c_int
        L.pf_sched_partition.argtypes = [POINTER(c_int), c_int, POINTER(c_int), c_int, c_int, c_int, POINTER(c_int)]
        L.pf_sched_destroy.restype = None
        L.pf_sched_destroy.argtypes = [c_void_p]
        L.pf_embedder_floats.restype = c_size_t
        L.pf_embedder_floats.argtypes = [POINTER(PfEmbedConfig)]
        L.pf_embedder_create.restype = c_int
        L.pf_embedder_create.argtypes = [POINTER(c_void_p), c_void_p, c_size_t, POINTER(PfEmbedConfig)]
        L.pf_embedder_forward.restype = c_int
        L.pf_embedder_forward.argtypes = [c_void_p, c_void_p, c_void_p, c_void_p, c_void_p, c_int, c_void_p, c_void_p,
                                          c_int, c_int, c_int, c_void_p]
        L.pf_embedder_last_launch_count.restype = c_longlong
        L.pf_embedder_last_launch_count.argtypes = [c_void_p]
        L.pf_embedder_destroy.restype = None
        L.pf_embedder_destroy.argtypes = [c_void_p]
        L.pf_extra_msa_block_floats.restype = c_size_t
        L.pf_extra_msa_block_floats.argtypes = [POINTER(PfExtraConfig)]
        L.pf_extra_msa_create.restype = c_int
        L.pf_extra_msa_create.argtypes = [POINTER(c_void_p), c_void_p, c_size_t, POINTER(PfExtraConfig)]
        L.pf_extra_msa_forward.restype = c_int
        L.pf_extra_msa_forward.argtypes = fwd + [c_int, c_void_p]
        L.pf_extra_msa_forward_substep.restype = c_int
        L.pf_extra_msa_forward_substep.argtypes = fwd + [c_int, c_int, c_void_p]
        L.pf_extra_msa_last_launch_count.restype = c_longlong
        L.pf_extra_msa_last_launch_count.argtypes = [c_void_p]
        L.pf_extra_msa_set_profiling.restype = c_int
        L.pf_extra_msa_set_profiling.argtypes = [c_void_p, c_int]
        L.pf_extra_msa_get_profile.restype = c_int
        L.pf_extra_msa_get_profile.argtypes = [c_void_p, c_int, POINTER(c_longlong), POINTER(ctypes.c_double),
                                               POINTER(ctypes.c_double), POINTER(ctypes.c_double)]
        L.pf_extra_msa_destroy.restype = None
        L.pf_extra_msa_destroy.argtypes = [c_void_p]
        L.pf_evoformer_forward_recycled.restype = c_int
        L.pf_evoformer_forward_recycled.argtypes = [c_void_p] * 14 + [c_int] * 7 + [c_void_p]
        L.pf_embedder_forward_extra.restype = c_int
        L.pf_embedder_forward_extra.argtypes = [c_void_p, c_void_p, c_void_p, c_int, c_int, c_int, c_void_p]
        L.pf_structure_floats.restype = c_size_t
        L.pf_structure_floats.argtypes = [POINTER(PfStructConfig)]
        L.pf_structure_create.restype = c_int
        L.pf_structure_create.argtypes = [POINTER(c_void_p), c_void_p, c_size_t, POINTER(PfStructConfig)]
        L.pf_structure_forward.restype = c_int
        L.pf_structure_forward.argtypes = [c_void_p] * 4 + [c_int] * 4 + [c_void_p] * 7
        L.pf_heads_forward.restype = c_int
        L.pf_heads_forward.argtypes = [c_void_p] * 3 + [c_int] * 3 + [c_void_p] * 4
        L.pf_plddt_forward_static.restype = c_int
        L.pf_plddt_forward_static.argtypes = [c_void_p, c_void_p, c_int, c_void_p, c_void_p]
        L.pf_structure_last_launch_count.restype = c_longlong
        L.pf_structure_last_launch_count.argtypes = [c_void_p]
        L.pf_structure_destroy.restype = None
        L.pf_structure_destroy.argtypes = [c_void_p]
        L.pf_fold_forward.restype = c_int
        L.pf_fold_forward.argtypes = [c_void_p] * 15 + [c_int] * 8 + [c_void_p] * 6
        _lib = L
    return _lib


def _check(status: int):
    if status != PF_OK:
        raise PfError(status, lib().pf_last_error().decode())


def _ptr(t):
    """Device/host pointer of a torch tensor, numpy array or raw int."""
    if t is None:
        return None
    if isinstance(t, int):
        return t
    if isinstance(t, np.ndarray):
        return t.ctypes.data
    return t.data_ptr()


def make_config(n_blocks_max: int, dtype: int = PF_BF16, c_m=256, c_z=128, heads_msa=8, heads_pair=4, head_dim=32,
                c_opm=32, c_tri=128, transition_n=4) -> PfConfig:
    return PfConfig(c_m, c_z, heads_msa, heads_pair, head_dim, c_opm, c_tri, transition_n, n_blocks_max, dtype)


def pf_evoformer_block_floats(cfg: PfConfig) -> int:
    return int(lib().pf_evoformer_block_floats(byref(cfg)))


class Evoformer:
    """Handle wrapper: pf_evoformer_create / forward / forward_substep / forward_host / destroy."""

    def __init__(self, weights_blob: np.ndarray, cfg: PfConfig):
        blob = np.ascontiguousarray(weights_blob, dtype=np.float32)
        self._h = c_void_p()
        self.cfg = cfg
        _check(lib().pf_evoformer_create(byref(self._h), blob.ctypes.data, blob.size, byref(cfg)))

    def _stream(self, stream):
        if stream is None:
            import torch
            return torch.cuda.current_stream().cuda_stream
        return stream

    def forward(self, msa, pair, seq_mask, msa_mask, n_blocks: int, stream=None):
        B, S, N = msa.shape[0], msa.shape[1], msa.shape[2]
        _check(lib().pf_evoformer_forward(self._h, _ptr(msa), _ptr(pair), _ptr(seq_mask), _ptr(msa_mask),
                                          B, S, N, n_blocks, self._stream(stream)))

    def forward_substep(self, msa, pair, seq_mask, msa_mask, block: int, substep: int, stream=None):
        B, S, N = msa.shape[0], msa.shape[1], msa.shape[2]
        _check(lib().pf_evoformer_forward_substep(self._h, _ptr(msa), _ptr(pair), _ptr(seq_mask), _ptr(msa_mask),
                                                  B, S, N, block, substep, self._stream(stream)))

    def forward_host(self, msa, pair, seq_mask, msa_mask, n_blocks: int, stream=None):
        B, S, N = msa.shape[0], msa.shape[1], msa.shape[2]
        _check(lib().pf_evoformer_forward_host(self._h, _ptr(msa), _ptr(pair), _ptr(seq_mask), _ptr(msa_mask),
                                               B, S, N, n_blocks, self._stream(stream)))

    def workspace_bytes(self, B: int, S: int, N: int) -> int:
        return int(lib().pf_evoformer_workspace_bytes(self._h, B, S, N))

    def set_profiling(self, enable: bool):
        _check(lib().pf_evoformer_set_profiling(self._h, 1 if enable else 0))

    def get_profile(self) -> dict:
        """{kind name: {"launches", "ms", "flops", "bytes"}} since set_profiling(True)."""
        out = {}
        for k in range(lib().pf_evoformer_profile_kinds()):
            n, ms, fl, by = c_longlong(), ctypes.c_double(), ctypes.c_double(), ctypes.c_double()
            _check(lib().pf_evoformer_get_profile(self._h, k, byref(n), byref(ms), byref(fl), byref(by)))
            out[lib().pf_evoformer_profile_name(k).decode()] = {
                "launches": n.value, "ms": ms.value, "flops": fl.value, "bytes": by.value}
        return out

    def get_profile_records(self) -> list:
        """[(kind name, ms, flops, bytes)] of every launch since set_profiling(True), in launch order."""
        out = []
        for i in range(int(lib().pf_evoformer_profile_records(self._h))):
            k, ms, fl, by = c_int(), ctypes.c_double(), ctypes.c_double(), ctypes.c_double()
            _check(lib().pf_evoformer_get_profile_record(self._h, i, byref(k), byref(ms), byref(fl), byref(by)))
            out.append((lib().pf_evoformer_profile_name(k.value).decode(), ms.value, fl.value, by.value))
        return out

    def last_launch_count(self) -> int:
        return int(lib().pf_evoformer_last_launch_count(self._h))

    def close(self):
        if self._h:
            lib().pf_evoformer_destroy(self._h)
            self._h = c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def make_extra_config(n_blocks_max: int, c_e=64, c_z=128, heads_msa=8, heads_pair=4, head_dim_pair=32, c_opm=32, c_tri=128,
                      transition_n=4) -> PfExtraConfig:
    return PfExtraConfig(c_e, c_z, heads_msa, heads_pair, head_dim_pair, c_opm, c_tri, transition_n, n_blocks_max)


class ExtraMsaStack:
    """pf_extra_msa_* wrapper (pointers and sizes only)."""

    def __init__(self, weights_blob: np.ndarray, cfg: PfExtraConfig):
        blob = np.ascontiguousarray(weights_blob, dtype=np.float32)
        self._x = c_void_p()
        self.cfg = cfg
        _check(lib().pf_extra_msa_create(byref(self._x), blob.ctypes.data, blob.size, byref(cfg)))

    @staticmethod
    def _stream(stream):
        if stream is None:
            import torch
            return torch.cuda.current_stream().cuda_stream
        return stream

    def forward(self, extra_msa, pair, seq_mask, extra_msa_mask, n_blocks: int, stream=None):
        B, S, N = extra_msa.shape[0], extra_msa.shape[1], extra_msa.shape[2]
        _check(lib().pf_extra_msa_forward(self._x, _ptr(extra_msa), _ptr(pair), _ptr(seq_mask), _ptr(extra_msa_mask),
                                          B, S, N, n_blocks, self._stream(stream)))

    def forward_substep(self, extra_msa, pair, seq_mask, extra_msa_mask, block: int, substep: int, stream=None):
        B, S, N = extra_msa.shape[0], extra_msa.shape[1], extra_msa.shape[2]
        _check(lib().pf_extra_msa_forward_substep(self._x, _ptr(extra_msa), _ptr(pair), _ptr(seq_mask), _ptr(extra_msa_mask),
                                                  B, S, N, block, substep, self._stream(stream)))

    def set_profiling(self, enable: bool):
        _check(lib().pf_extra_msa_set_profiling(self._x, 1 if enable else 0))

    def get_profile(self) -> dict:
        out = {}
        for k in range(lib().pf_evoformer_profile_kinds()):
            n, ms, fl, by = c_longlong(), ctypes.c_double(), ctypes.c_double(), ctypes.c_double()
            _check(lib().pf_extra_msa_get_profile(self._x, k, byref(n), byref(ms), byref(fl), byref(by)))
            out[lib().pf_evoformer_profile_name(k).decode()] = {
                "launches": n.value, "ms": ms.value, "flops": fl.value, "bytes": by.value}
        return out

    def last_launch_count(self) -> int:
        return int(lib().pf_extra_msa_last_launch_count(self._x))

    def close(self):
        if self._x:
            lib().pf_extra_msa_destroy(self._x)
            self._x = c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def make_embed_config(c_m=256, c_z=128, tf_dim=22, msa_dim=49, max_relpos=32, n_dist_bins=15, first_break=3.25,
                      last_break=20.75, extra_dim=25, c_e=64) -> PfEmbedConfig:
    return PfEmbedConfig(c_m, c_z, tf_dim, msa_dim, max_relpos, n_dist_bins, first_break, last_break, extra_dim, c_e)


class Embedder:
    """pf_embedder_* wrapper: input + recycling embedders (pointers and sizes only)."""

    def __init__(self, weights_blob: np.ndarray, cfg: PfEmbedConfig):
        blob = np.ascontiguousarray(weights_blob, dtype=np.float32)
        self._e = c_void_p()
        self.cfg = cfg
        _check(lib().pf_embedder_create(byref(self._e), blob.ctypes.data, blob.size, byref(cfg)))

    def forward(self, target_feat, residue_index, msa_feat, x_prev, has_prev: bool, msa, pair, stream=None):
        B, S, N = msa.shape[0], msa.shape[1], msa.shape[2]
        if stream is None:
            import torch
            stream = torch.cuda.current_stream().cuda_stream
        _check(lib().pf_embedder_forward(self._e, _ptr(target_feat), _ptr(residue_index), _ptr(msa_feat), _ptr(x_prev),
                                         1 if has_prev else 0, _ptr(msa), _ptr(pair), B, S, N, stream))

    def forward_extra(self, extra_msa_feat, extra_msa, stream=None):
        B, S_e, N = extra_msa.shape[0], extra_msa.shape[1], extra_msa.shape[2]
        if stream is None:
            import torch
            stream = torch.cuda.current_stream().cuda_stream
        _check(lib().pf_embedder_forward_extra(self._e, _ptr(extra_msa_feat), _ptr(extra_msa), B, S_e, N, stream))

    def last_launch_count(self) -> int:
        return int(lib().pf_embedder_last_launch_count(self._e))

    def close(self):
        if self._e:
            lib().pf_embedder_destroy(self._e)
            self._e = c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def forward_recycled(evo: "Evoformer", emb: Embedder, target_feat, residue_index, msa_feat, x_prev, msa, pair, seq_mask,
                     msa_mask, n_blocks: int, n_cycles: int, stream=None, extra: "ExtraMsaStack" = None, extra_msa_feat=None,
                     extra_msa=None, extra_msa_mask=None, n_extra_blocks: int = 0):
    """pf_evoformer_forward_recycled: n_cycles x (embedders [, extra-MSA stack], trunk); msa / pair receive the result."""
    B, S, N = msa.shape[0], msa.shape[1], msa.shape[2]
    S_e = extra_msa.shape[1] if extra is not None else 0
    _check(lib().pf_evoformer_forward_recycled(evo._h, emb._e, extra._x if extra is not None else None, _ptr(target_feat),
                                               _ptr(residue_index), _ptr(msa_feat), _ptr(x_prev), _ptr(extra_msa_feat),
                                               _ptr(extra_msa), _ptr(extra_msa_mask), _ptr(msa), _ptr(pair), _ptr(seq_mask),
                                               _ptr(msa_mask), B, S, S_e, N, n_blocks, n_extra_blocks, n_cycles,
                                               evo._stream(stream)))


def make_struct_config(c_m=256, c_z=128, c_s=384, heads=12, c_ipa=16, n_qp=4, n_pv=8, n_layers=8, c_resnet=128, n_torsion=7,
                       n_dist_bins=64, n_msa_classes=23, n_lddt_bins=50, c_lddt=128, n_pae_bins=64, n_resolved=37,
                       pos_scale=10.0) -> PfStructConfig:
    return PfStructConfig(c_m, c_z, c_s, heads, c_ipa, n_qp, n_pv, n_layers, c_resnet, n_torsion, n_dist_bins, n_msa_classes,
                          n_lddt_bins, c_lddt, n_pae_bins, n_resolved, pos_scale)


class StructureModule:
    """pf_structure_* / pf_heads_forward wrapper (pointers and sizes only)."""

    def __init__(self, weights_blob: np.ndarray, cfg: PfStructConfig):
        blob = np.ascontiguousarray(weights_blob, dtype=np.float32)
        self._s = c_void_p()
        self.cfg = cfg
        _check(lib().pf_structure_create(byref(self._s), blob.ctypes.data, blob.size, byref(cfg)))

    @staticmethod
    def _stream(stream):
        if stream is None:
            import torch
            return torch.cuda.current_stream().cuda_stream
        return stream

    def forward(self, msa, pair, seq_mask, n_layers=None, s_out=None, frames_out=None, x_out=None, alpha_out=None,
                plddt_out=None, resolved_out=None, stream=None):
        B, S, N = msa.shape[0], msa.shape[1], msa.shape[2]
        _check(lib().pf_structure_forward(self._s, _ptr(msa), _ptr(pair), _ptr(seq_mask), B, S, N,
                                          self.cfg.n_layers if n_layers is None else n_layers, _ptr(s_out), _ptr(frames_out),
                                          _ptr(x_out), _ptr(alpha_out), _ptr(plddt_out), _ptr(resolved_out), self._stream(stream)))

    def heads(self, msa, pair, distogram_out=None, masked_msa_out=None, pae_out=None, stream=None):
        ref = msa if msa is not None else pair
        B, N = ref.shape[0], ref.shape[2]
        S = msa.shape[1] if msa is not None else 1
        _check(lib().pf_heads_forward(self._s, _ptr(msa), _ptr(pair), B, S, N, _ptr(distogram_out), _ptr(masked_msa_out),
                                      _ptr(pae_out), self._stream(stream)))

    def plddt_static(self, s, plddt_out, stream=None):
        """pf_plddt_forward_static: H.3 on s[..., c_s] with no allocation (file-scope device scratch, shared by all calls)."""
        rows = 1
        for d in s.shape[:-1]:
            rows *= int(d)
        _check(lib().pf_plddt_forward_static(self._s, _ptr(s), rows, _ptr(plddt_out), self._stream(stream)))

    def last_launch_count(self) -> int:
        return int(lib().pf_structure_last_launch_count(self._s))

    def close(self):
        if self._s:
            lib().pf_structure_destroy(self._s)
            self._s = c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def fold_forward(evo: "Evoformer", emb: Embedder, sm: StructureModule, target_feat, residue_index, msa_feat, x_prev0, msa,
                 pair, seq_mask, msa_mask, n_blocks: int, n_cycles: int, x_cycles_out, n_layers=None, s_out=None,
                 frames_out=None, alpha_out=None, plddt_out=None, stream=None, extra: "ExtraMsaStack" = None,
                 extra_msa_feat=None, extra_msa=None, extra_msa_mask=None, n_extra_blocks: int = 0):
    """pf_fold_forward: n_cycles x (embedders fed with the previous cycle's positions [, extra-MSA stack], trunk, structure
    module); msa / pair receive the last trunk output, x_cycles_out [n_cycles,B,N,3] the positions after every cycle."""
    B, S, N = msa.shape[0], msa.shape[1], msa.shape[2]
    S_e = extra_msa.shape[1] if extra is not None else 0
    _check(lib().pf_fold_forward(evo._h, emb._e, extra._x if extra is not None else None, sm._s, _ptr(target_feat),
                                 _ptr(residue_index), _ptr(msa_feat), _ptr(x_prev0), _ptr(extra_msa_feat), _ptr(extra_msa),
                                 _ptr(extra_msa_mask), _ptr(msa), _ptr(pair), _ptr(seq_mask), _ptr(msa_mask), B, S, S_e, N,
                                 n_blocks, n_extra_blocks, n_cycles, sm.cfg.n_layers if n_layers is None else n_layers,
                                 _ptr(x_cycles_out), _ptr(s_out), _ptr(frames_out), _ptr(alpha_out), _ptr(plddt_out),
                                 evo._stream(stream)))


class Scheduler:
    """pf_sched_* wrapper: length-bucketing batch scheduler."""

    def __init__(self, buckets, mem_budget_bytes: int, S: int):
        arr = (c_int * len(buckets))(*buckets)
        self._s = c_void_p()
        st = lib().pf_sched_create(byref(self._s), arr, len(buckets), mem_budget_bytes, S)
        if st != PF_OK:
            raise PfError(st, "pf_sched_create")

    def add(self, protein_id: int, length: int):
        st = lib().pf_sched_add(self._s, protein_id, length)
        if st != PF_OK:
            raise PfError(st, f"pf_sched_add(id={protein_id}, length={length})")

    def next_batch(self, cap: int = 4096):
        ids = (c_int * cap)()
        lens = (c_int * cap)()
        bucket = c_int()
        n = lib().pf_sched_next_batch(self._s, ids, lens, cap, byref(bucket))
        if n < 0:
            raise PfError(1, "pf_sched_next_batch")
        if n == 0:
            return None
        return list(ids[:n]), list(lens[:n]), bucket.value

    def batches(self, cap: int = 4096):
        while True:
            b = self.next_batch(cap)
            if b is None:
                return
            yield b

    def close(self):
        if self._s:
            lib().pf_sched_destroy(self._s)
            self._s = c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def bytes_per_protein(bucket: int, S: int) -> int:
    return int(lib().pf_sched_bytes_per_protein(bucket, S))


def sched_cost(bucket: int, S: int) -> float:
    return float(lib().pf_sched_cost(bucket, S))


def partition(lengths, buckets, S: int, world: int):
    """pf_sched_partition: rank of every protein (replicas-only multi-GPU: the protein LIST is sharded, no collective)."""
    n = len(lengths)
    la = (c_int * max(n, 1))(*[int(x) for x in lengths])
    ba = (c_int * len(buckets))(*[int(b) for b in buckets])
    out = (c_int * max(n, 1))()
    st = lib().pf_sched_partition(la, n, ba, len(buckets), S, world, out)
    if st != PF_OK:
        raise PfError(st, "pf_sched_partition")
    return [int(out[i]) for i in range(n)]
