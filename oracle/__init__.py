"""fp64 CPU oracle — TEST INFRASTRUCTURE (see oracle/lpm_oracle.c header)."""
