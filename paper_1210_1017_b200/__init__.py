"""B200-native SPH hot path of arXiv 1210.1017 (Valdez-Balderas et al.).

The package holds three things only:

* ``csrc/``      - hand-written sm_100a CUDA kernels and the C-ABI library
                   ``libsph_b200.so`` declared in ``include/sph_b200.h``;
* ``binding``    - a thin ctypes binding with the same names as the C ABI
                   (argument marshalling only; every step runs in the kernels);
* ``workloads``  - seeded synthetic input generators (no method arithmetic).

Nothing here imports ``oracle/`` and ``oracle/`` imports nothing from here.
Importing this package is cheap; ``binding`` is imported on first use and
fails loudly when the CUDA library has not been built.
"""

__all__ = ["binding", "workloads", "build"]
__version__ = "0.1.0"
