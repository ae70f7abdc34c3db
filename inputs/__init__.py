"""Seeded synthetic input generators shared by the oracle's tests, the CUDA path's tests and bench.py.
Holds none of the imaging method's arithmetic."""
