"""Brute-force fp64 CPU oracle.  TEST INFRASTRUCTURE, NOT THE PRODUCT (see hcgrid_oracle.h)."""
