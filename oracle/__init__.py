"""float64 CPU oracle (test infrastructure only; see oracle/lcf_oracle.c)."""
