"""CPU oracle of the SCAPE step — TEST INFRASTRUCTURE ONLY (see scape_oracle.cpp)."""
