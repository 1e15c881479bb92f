"""CPU oracle of the piMPC ADMM iteration -- test infrastructure only (see pimpc_oracle.c)."""
