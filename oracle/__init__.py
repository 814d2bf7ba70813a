"""CPU oracle (test infrastructure only; see oracle/qmc_oracle.h)."""
