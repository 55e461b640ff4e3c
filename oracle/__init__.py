"""FP64 CPU oracle (test infrastructure only; see oracle/sp2_oracle.py)."""
