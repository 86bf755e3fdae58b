"""CPU oracle (test infrastructure). See oracle/afqmc_oracle.py. Never imported by the product path."""
