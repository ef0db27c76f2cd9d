"""CPU oracle of the CheFSI hot path -- test infrastructure, not product (see chefsi_oracle.c)."""
