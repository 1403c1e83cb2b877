"""CPU oracle for the CGKS-5 / S2O4 hot path.  TEST INFRASTRUCTURE ONLY (see cgks_ref.h)."""
