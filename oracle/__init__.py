"""ORACLE - test infrastructure only. See oracle/reference.py and oracle/ig_oracle.c."""
