"""fp64 CPU oracle -- TEST INFRASTRUCTURE, NOT THE PRODUCT (see smre_oracle.c header)."""
