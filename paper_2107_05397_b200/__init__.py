"""B200-native Striped/Hybrid UniFrac all-pairs distance (arXiv 2107.05397 hot path).

The package holds only what the path needs:

* ``csrc/``     -- the sm_100a CUDA kernels and the C-ABI (``include/unifrac_b200.h``)
* ``binding``   -- thin ctypes binding with the same names (argument marshalling only)
* ``build``     -- the in-tree nvcc build step
* ``synth``     -- seeded synthetic input generators (no UniFrac arithmetic); the only module
                   shared by the CUDA path's tests/bench and the CPU oracle's tests.

Nothing here imports ``oracle/``; importing the package does not load the CUDA library
(``binding.load()`` does, and fails loudly if the library is missing).
"""

__all__ = ["binding", "build", "synth"]
