"""fp64 CPU oracle (test infrastructure only -- see rfa_oracle.py)."""
