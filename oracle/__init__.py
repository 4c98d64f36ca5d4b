"""CPU fp64 oracle of the Hermite hot path -- TEST INFRASTRUCTURE, NOT THE PRODUCT (see nbody_oracle.c header)."""
