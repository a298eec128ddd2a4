"""FP64 CPU oracle (test infrastructure; see oracle/mlmd_ref.c for what it computes)."""
