"""CPU oracle package — TEST INFRASTRUCTURE ONLY (see t_oracle.py header)."""
