"""CPU oracle (TEST INFRASTRUCTURE — see oracle/dit_oracle.py header)."""
