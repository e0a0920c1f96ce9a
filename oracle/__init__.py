"""CPU oracle of the Independent algorithm -- TEST INFRASTRUCTURE ONLY (see oracle/necsim_oracle.c)."""
