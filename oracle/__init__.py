"""CPU oracle -- TEST INFRASTRUCTURE, not the product. See oracle/oracle.c."""
