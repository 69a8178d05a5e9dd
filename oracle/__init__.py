"""fp64 CPU oracle for the radiation detector -- TEST INFRASTRUCTURE ONLY (see rad_oracle.c)."""
