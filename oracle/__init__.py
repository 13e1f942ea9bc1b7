"""CPU oracle: test infrastructure only (see oracle/cdz_oracle.h)."""
