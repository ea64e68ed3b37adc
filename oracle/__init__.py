"""CPU oracle for the Ozaki-II DGEMM path -- test infrastructure, not product (see ozaki2_oracle.c)."""
