"""CPU oracle (test infrastructure only). See oracle/bh_oracle.c and oracle/bh_oracle.py."""
