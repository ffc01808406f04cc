"""fp64 CPU oracle (test infrastructure; see oracle/qcf_oracle.py header)."""
from .qcf_oracle import *  # noqa: F401,F403
