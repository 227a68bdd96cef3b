"""Seeded synthetic input generators shared by the tests, bench.py and the oracle's pins (no loss arithmetic lives here;
neither the CUDA binding nor the oracle is imported)."""
