"""fp64 CPU oracle (test infrastructure only; see evoformer_ref.py header)."""
from .evoformer_ref import *  # noqa: F401,F403
from . import evoformer_ref  # noqa: F401
from . import evoformer_sampled, embed_ref, extra_msa_ref, structure_ref  # noqa: F401
from .evoformer_sampled import Rounding, substep_at, substep_all, block_all  # noqa: F401
