"""ORACLE — test infrastructure only (see homg_oracle.cpp).  Never imported by the product path."""
