"""CPU FP64 oracle (test infrastructure only; see zfac_oracle.py header)."""
