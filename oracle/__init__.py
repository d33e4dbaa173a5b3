"""CPU oracle (test infrastructure only; see spense_oracle.py header)."""
