"""CPU oracle -- test infrastructure only (see oracle/bit1_oracle.c header)."""
