"""CPU oracle (TEST INFRASTRUCTURE, not product). See oracle/ozfft_oracle.c."""
