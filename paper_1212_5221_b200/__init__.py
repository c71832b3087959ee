"""B200-native SU(3) lattice gauge fixing (checkerboard sweep), arxiv/paper_1212_5221.

The package is a thin binding over ``libgf.so`` (hand-written sm_100a CUDA behind the
C ABI declared in ``include/gf.h``).  Importing the package does not load the library;
``paper_1212_5221_b200.gf`` does, and fails loudly when it is missing.
``paper_1212_5221_b200.inputs`` holds the seeded synthetic-lattice generators (no method
arithmetic) that both the tests of the CPU oracle and the CUDA path draw their inputs from.
"""

__all__ = ["gf", "inputs", "build"]
