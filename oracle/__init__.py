"""CPU fp64 oracle of the submatrix sign-function method -- test infrastructure only."""
