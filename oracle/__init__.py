"""CPU oracle package: test infrastructure only (see lbm_oracle.cpp header)."""
