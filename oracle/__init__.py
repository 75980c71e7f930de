"""CPU oracle for Sketch&Walk Attention -- test infrastructure only (see sw_oracle.py)."""
