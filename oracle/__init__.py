"""CPU oracle for the FDAS hot path -- test infrastructure only (see fdas_oracle.c header)."""
