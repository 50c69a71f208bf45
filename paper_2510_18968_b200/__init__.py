"""paper_2510_18968_b200 -- B200-native resistive GRMHD IMEX-RK2 step.

The package holds only what the hot path needs:

* ``csrc/``       hand-written sm_100a CUDA kernels and the C-ABI (``include/rgrmhd.h``)
* ``binding.py``  thin ctypes binding with the same names (argument marshalling only)
* ``workloads.py`` seeded synthetic input generators (no method arithmetic; shared with
  the oracle tests)
* ``build.py``    in-tree nvcc build of ``librgrmhd.so``

Nothing here imports ``oracle/``; importing the package does not load the CUDA library
(``binding.load()`` does, and fails loudly when it is missing).
"""

__all__ = ["binding", "workloads", "build"]
