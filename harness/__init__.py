"""Seeded synthetic-input generators (shared by the oracle-side tests and the CUDA path; no method arithmetic)."""
