"""CPU ORACLE package — test infrastructure, not the product (see oracle/nfs_oracle.c header)."""
