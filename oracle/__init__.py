"""CPU oracle — test infrastructure only (see legs_oracle.cpp header)."""
