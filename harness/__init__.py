"""harness — seeded synthetic input generators shared by the tests, bench.py and smoke().

Holds none of the method's arithmetic (no projection, interpolation or TDI): orbit tables, waveforms and workload
descriptors only.  Both the product's callers and the oracle's callers import it; neither oracle/ nor
paper_2204_06633_b200/ does.
"""
