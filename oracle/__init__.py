"""FDAS oracle package -- test infrastructure only (see oracle/fdas_oracle.py)."""
