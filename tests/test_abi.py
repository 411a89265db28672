"""The C-ABI library loads and exports every symbol include/pf_evoformer.h declares (no GPU needed)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def built_lib():
    from paper_2111_06340_b200 import build
    return build.build()


def test_header_symbols_exported(built_lib):
    hdr = open(os.path.join(ROOT, "include", "pf_evoformer.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(pf_[a-z0-9_]+)\s*\(", hdr))
    assert {"pf_evoformer_create", "pf_evoformer_forward", "pf_sched_next_batch"} <= declared
    L = ctypes.CDLL(built_lib)
    for name in sorted(declared):
        assert hasattr(L, name), f"{name} declared in the header but not exported"
    import paper_2111_06340_b200 as pf
    assert declared == set(pf.EXPORTED_SYMBOLS)


def test_block_floats_matches_appendix_b(built_lib):
    import paper_2111_06340_b200 as pf
    import pf_synth as ps
    assert pf.pf_evoformer_block_floats(pf.make_config(1)) == ps.block_floats() == 1829952


def test_no_oracle_import_in_product():
    """The product path must never route through the oracle."""
    pkg = os.path.join(ROOT, "paper_2111_06340_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", src, flags=re.M), f
    for dirpath, _, files in os.walk(os.path.join(ROOT, "oracle")):
        for f in files:
            if f.endswith(".py"):
                assert "paper_2111_06340_b200" not in re.sub(r'""".*?"""', "", open(os.path.join(dirpath, f)).read(), flags=re.S), f
