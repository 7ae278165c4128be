"""ORACLE -- test infrastructure only (see evis_oracle.c).  Never imported by the product path."""
