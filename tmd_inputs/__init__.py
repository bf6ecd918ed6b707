"""Seeded synthetic inputs and data-layout definitions for TPC track-model decoding.

This package serves BOTH the CPU oracle (``oracle/``) and the CUDA library
(``paper_2411_02206_b200/``).  It holds no arithmetic of the method itself
(no track model, no residual coding, no prefix sums of the codec): only

* ``layout``   -- numpy dtypes / containers for the compressed SoA and the 16-byte cluster record
                  (SURVEY.md §8(b), §8(c)-C2),
* ``geometry`` -- the synthetic pad-plane tables, built in double and cast to fp32,
* ``physical`` -- helix event generator in the cluster domain (to be encoded by the oracle encoder in tests),
* ``compressed`` -- counter-based generator that draws time frames directly in the compressed domain
                  (what ``bench.py`` decodes; device-agnostic integer torch ops).
"""
from .layout import CLUSTER_DTYPE, Compressed, N_ROWS, N_AZ, N_SIDES  # noqa: F401
from .geometry import Geometry, build_geometry  # noqa: F401
