"""CPU oracle (test infrastructure only). See oracle/ulens_oracle.c and oracle/oracle.py."""
