"""CPU oracle package -- TEST INFRASTRUCTURE, not the product (see oracle/tso.h)."""
