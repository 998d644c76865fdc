"""Seeded synthetic input generators shared by oracle-side and CUDA-side tests (no method arithmetic)."""
