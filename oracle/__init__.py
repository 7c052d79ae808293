"""CPU oracle for the FHGS hot path -- test infrastructure only (see fhgs_oracle.c header)."""
