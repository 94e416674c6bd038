"""CPU fp64 oracle (test infrastructure only; see oracle/omni_oracle.c header)."""
