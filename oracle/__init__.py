"""fp64 CPU oracle (test infrastructure only; see tts_oracle.py)."""
