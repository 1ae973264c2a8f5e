"""CPU fp64 oracle for SRA - test infrastructure only (see sra_oracle.py header)."""
