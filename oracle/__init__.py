"""CPU oracle (test infrastructure only; see df_oracle.py's header)."""
from .df_oracle import *  # noqa: F401,F403
