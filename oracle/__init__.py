"""float64 CPU oracle for the SF-TR projector pair -- test infrastructure only (see sf_oracle.c)."""
