"""CPU oracle (test infrastructure, not product code). See oracle/epic_oracle.py."""
