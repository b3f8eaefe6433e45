"""FP64 CPU oracle (test infrastructure only; see nolsm_oracle.py header)."""
from .nolsm_oracle import *  # noqa: F401,F403
