"""CPU oracle package: test infrastructure only (see mlip_oracle.py header)."""
