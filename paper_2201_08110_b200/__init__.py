"""B200-native ANI-2x energy+force hot path of NNP/MM (arXiv 2201.08110).

The product is the C-ABI library declared in ``include/nnp.h`` (CUDA kernels for
sm_100a under ``csrc/``) plus the thin ctypes binding in ``binding.py``.
``workloads.py`` holds the seeded synthetic input generators only (no method
arithmetic); it is the one module shared by the tests of the CUDA path and of
the CPU oracle under ``oracle/``.

Nothing here imports ``oracle/`` and there is no CPU fallback: using the
binding without the compiled ``libnnp_b200.so`` raises.
"""

__all__ = ["workloads", "binding"]
