"""CPU oracle for the FDTD Yee update -- TEST INFRASTRUCTURE, never imported by the product path."""
