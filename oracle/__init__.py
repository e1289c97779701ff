"""CPU oracle (test infrastructure only; see qs_oracle.py header)."""
