"""Oracle: test infrastructure only (see oracle/kbmod_oracle.c header)."""
