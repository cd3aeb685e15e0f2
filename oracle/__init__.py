"""CPU oracle of the submatrix method -- test infrastructure only (see submatrix_oracle.c)."""
