"""float64 CPU oracle (test infrastructure only; see himuon_oracle.py header)."""
