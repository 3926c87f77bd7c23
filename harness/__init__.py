"""Seeded synthetic input generators shared by the CUDA path's callers (tests, bench.py, smoke) and the oracle's
callers.  This package holds none of the method's arithmetic and imports neither `paper_2501_00675_b200` nor
`oracle`: it exists so that both sides see the same bytes."""
