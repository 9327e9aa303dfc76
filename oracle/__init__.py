"""CPU double-precision oracle for the CWO++ hot path -- test infrastructure only (see cwo_oracle.c)."""
