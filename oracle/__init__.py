"""CPU oracle (test infrastructure only; see lya_oracle.c header)."""
