"""CPU oracle of the diffHydro coupled step -- TEST INFRASTRUCTURE, not the product (see dh_oracle.cpp)."""
