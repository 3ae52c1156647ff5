"""Test infrastructure only: the fp64 CPU oracle.  See mm_oracle.py."""
