"""CPU oracle of the Splotch rendering path -- test infrastructure only (see splotch_oracle.c)."""
