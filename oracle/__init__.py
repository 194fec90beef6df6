"""CPU oracle (test infrastructure only -- see oracle/fdtd_oracle.c header)."""
