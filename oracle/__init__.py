"""float64 CPU oracle (test infrastructure; see oracle/block_causal.py header)."""
