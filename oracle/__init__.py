"""CPU oracle package -- test infrastructure only (see vibe_oracle.py header)."""
