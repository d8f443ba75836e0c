"""B200-native MaxSim scoring (TileMaxSim hot path): C-ABI CUDA library + thin Python binding.

``from paper_2606_26439_b200 import tms`` gives the binding (same names as include/tms.h);
``paper_2606_26439_b200.synth`` holds the seeded input generators.  Importing this package never
loads the oracle and never falls back to a CPU path: binding calls raise if libtms.so is missing.
"""
__all__ = ["tms", "synth", "accounting"]
