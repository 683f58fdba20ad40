"""CPU oracle package (test infrastructure only; see jerk_oracle.py header)."""
