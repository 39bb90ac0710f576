"""CPU oracle for the StePS hot path -- TEST INFRASTRUCTURE ONLY (see steps_oracle.c)."""
