"""ORACLE package -- test infrastructure only (see tdde_oracle.py header)."""
