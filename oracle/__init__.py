"""float64 CPU oracle for the DPSR layer -- TEST INFRASTRUCTURE ONLY (see dpsr_oracle.c header)."""
