"""fp64 CPU oracle (test infrastructure only; see evoformer_ref.py header)."""
from .evoformer_ref import *  # noqa: F401,F403
from . import evoformer_ref  # noqa: F401
