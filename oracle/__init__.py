"""fp64 CPU oracle of the ODISSEO hot path -- test infrastructure only (see oracle.py)."""
