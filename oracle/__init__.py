"""CPU fp64 oracle (test infrastructure only; see gecc_oracle.py).  Never imported by the product path."""
