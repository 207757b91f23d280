"""fp64 CPU oracle — test infrastructure only (see te_oracle.py header)."""
