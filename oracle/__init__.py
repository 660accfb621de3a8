"""fp64 CPU oracle (TEST INFRASTRUCTURE; see oracle/hb_oracle.c header)."""
from .oracle import *  # noqa: F401,F403
