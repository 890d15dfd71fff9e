"""fp64 CPU oracle (test infrastructure, not the product). See md_oracle.c."""
