"""CPU fp64 oracle of the hot path -- TEST INFRASTRUCTURE, NOT PRODUCT (see smlm_oracle.c)."""
