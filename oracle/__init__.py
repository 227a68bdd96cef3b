"""fp64 CPU oracle (test infrastructure only; see opd_oracle.py)."""
