"""CPU oracle (test infrastructure). See oracle/poisson_oracle.c and oracle/oracle.py."""
