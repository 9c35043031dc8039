"""CPU oracle for the wave2d ADI hot path.  Test infrastructure only -- see oracle/wave2d_oracle.c."""
