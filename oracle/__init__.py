"""CPU oracle package -- test infrastructure only (see pyr_oracle.c header)."""
