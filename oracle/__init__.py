"""CPU oracle for the BLINK hot path (test infrastructure only; see blink_oracle.c)."""
