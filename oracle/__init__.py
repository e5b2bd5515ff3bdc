"""CPU oracle for the GPipe hot path - TEST INFRASTRUCTURE (see gpipe_oracle.py header)."""
