"""CPU oracle -- test infrastructure only (see crf_oracle.c header)."""
