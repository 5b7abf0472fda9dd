"""Seeded synthetic input generators (BASELINE.json configs) shared by the CUDA path's harness and by the oracle's
tests.  A module of its own: it holds none of the method's arithmetic and imports neither the CUDA binding nor the oracle."""
