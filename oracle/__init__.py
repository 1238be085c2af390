"""CPU oracle of the ECHO RMHD step — test infrastructure only (see echo_oracle.cpp)."""
