"""CPU oracle for the Debye summation -- TEST INFRASTRUCTURE, not the product (see debye_oracle.c)."""
