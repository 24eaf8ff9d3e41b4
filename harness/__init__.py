"""Test and bench harness: seeded synthetic input generators shared by the CPU oracle's tests and the
CUDA path's tests / bench.  Holds none of the method's arithmetic and imports neither side."""
