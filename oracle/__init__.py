"""CPU oracle for the Wilson-Dirac matvec (test infrastructure only; see wd_oracle.c)."""
