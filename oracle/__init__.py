"""CPU oracle (test infrastructure only) -- see oracle/lrp_oracle.py."""
