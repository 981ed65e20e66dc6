"""CPU oracle of the MEG6 hot path (test infrastructure, not the product). See meg6_oracle.cpp."""
