"""FP64 CPU oracle (test infrastructure only; see oracle/wl_oracle.c header)."""
