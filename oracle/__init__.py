"""CPU oracle and exact references: test infrastructure (see oracle/pa_oracle.cpp header)."""
