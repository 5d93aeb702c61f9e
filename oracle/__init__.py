"""Float64 CPU oracle (test infrastructure only; see delta_oracle.py's header)."""
