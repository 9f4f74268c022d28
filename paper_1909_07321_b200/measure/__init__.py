"""Measurement utilities that sit beside the product library (bench.py uses them; the hot path does not)."""
