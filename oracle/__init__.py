"""CPU oracle of the particle-mesh-particle step -- test infrastructure only (see pm_oracle.c)."""
