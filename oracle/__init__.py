"""CPU oracle package (TEST INFRASTRUCTURE ONLY; see oracle/fe_oracle.c)."""
