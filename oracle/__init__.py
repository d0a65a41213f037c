"""fp64 CPU oracle of the plane-wise multi-view RL iteration.  TEST INFRASTRUCTURE -- see mvd_oracle.c."""
