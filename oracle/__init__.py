"""CPU oracle package.  TEST INFRASTRUCTURE ONLY -- see oracle/rmhd_oracle.cpp."""
