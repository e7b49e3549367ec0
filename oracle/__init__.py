"""fp64 CPU oracle of the Delphes-style detector response: TEST INFRASTRUCTURE ONLY (see pd_oracle.h)."""
