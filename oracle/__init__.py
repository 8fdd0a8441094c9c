"""CPU oracle (test infrastructure only) -- see tatrg_oracle.py."""
