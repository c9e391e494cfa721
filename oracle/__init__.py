"""CPU oracle (test infrastructure only; see fdd_oracle.py)."""
