"""CPU oracle for the ENUF path (test infrastructure only; see enuf_oracle.c)."""
