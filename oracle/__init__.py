"""ORACLE — test infrastructure only (see trace_oracle.py and brute_force.py).  Not part of the product path."""
