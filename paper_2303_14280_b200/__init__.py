"""snk — B200-native seminumerical exact-exchange (sn-K) build, arXiv 2303.14280 Sec. II D/E + App. A.

The package holds only what the hot path needs:
  * ``csrc/``     hand-written sm_100a CUDA + the C-ABI library (``include/snk.h``)
  * ``snk.py``    thin ctypes binding with the same names (argument marshalling only)
  * ``inputs.py`` seeded synthetic inputs (shared with the CPU oracle; no method arithmetic)
  * ``build.py``  nvcc build of ``libsnk.so`` (in-tree)

Importing the package does NOT load the CUDA library; ``snk.load()`` does, and fails
loudly when it is missing.  Nothing here imports ``oracle/``.
"""
__version__ = "0.1.0"
