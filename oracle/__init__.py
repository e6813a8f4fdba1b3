"""CPU oracle for the Omega(Delta; q, h, T) hot path.  TEST INFRASTRUCTURE, NOT THE PRODUCT (see fe_oracle.c)."""
