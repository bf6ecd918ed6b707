"""Synthetic "ALICE-like" pad-plane geometry.

The paper states no geometry (PAPER.md L70 says only "propagates it through the TPC"); these tables are this
build's reading: 36 sectors x 152 pad rows, 20-degree sectors, four pad regions.  They are built in double
precision and cast to fp32 once, then handed *identically* to the CPU oracle and to the CUDA library
(both receive them as inputs, neither recomputes them).
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np

from .layout import N_AZ, N_ROWS, N_SIDES

TAN10 = 0.17632698070846498            # tan(10 deg)
COS_A = np.float32(0.93969262078590838)  # cos(20 deg) -> 0x3f708fb2
SIN_A = np.float32(0.34202014332566873)  # sin(20 deg) -> 0x3eaf1d44
TF_NBINS = 14256                       # time bins per time frame (generator parameter only)

# (first row, last row, x of first row [cm], row pitch [cm], pad width [cm])
REGIONS = ((0, 62, 85.0, 0.75, 0.4), (63, 96, 135.0, 1.0, 0.6),
           (97, 126, 171.0, 1.2, 0.6), (127, 151, 209.0, 1.5, 0.6))


@dataclass(frozen=True)
class Geometry:
    n_az: int
    n_sides: int
    n_sectors_out: int
    n_rows: int
    cos_a: np.float32
    sin_a: np.float32
    row_x: np.ndarray         # f32[n_rows] cm
    row_padw: np.ndarray      # f32[n_rows] cm
    row_inv_padw: np.ndarray  # f32[n_rows] 1/cm
    row_npads: np.ndarray     # u16[n_rows], even
    row_x_f64: np.ndarray     # generator-side double copies
    row_padw_f64: np.ndarray

    @property
    def n_bins(self) -> int:
        return self.n_sectors_out * self.n_rows


def build_geometry(n_sectors_out: int = N_AZ * N_SIDES) -> Geometry:
    x = np.zeros(N_ROWS, dtype=np.float64)
    w = np.zeros(N_ROWS, dtype=np.float64)
    for r0, r1, x0, pitch, padw in REGIONS:
        r = np.arange(r0, r1 + 1)
        x[r] = x0 + pitch * (r - r0)
        w[r] = padw
    npads = (2 * np.floor(x * TAN10 / w)).astype(np.uint16)
    return Geometry(
        n_az=N_AZ, n_sides=N_SIDES, n_sectors_out=n_sectors_out, n_rows=N_ROWS,
        cos_a=COS_A, sin_a=SIN_A,
        row_x=x.astype(np.float32), row_padw=w.astype(np.float32),
        row_inv_padw=(1.0 / w).astype(np.float32), row_npads=npads,
        row_x_f64=x, row_padw_f64=w,
    )
