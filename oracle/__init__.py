"""CPU oracle (TEST INFRASTRUCTURE, not the product). See oracle/dse_oracle.c."""
