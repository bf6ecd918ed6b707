"""Adversarial compressed inputs: valid counts, arbitrary bytes in every value array (SURVEY.md §8(c)-C8 "adversarial").

Decoding is defined for any stream values (DESIGN.md §3 readings 15, 19), so the CUDA path must agree with the oracle
on these too.  No arithmetic of the method lives here: only seeded draws into the layout's arrays.
"""
from __future__ import annotations

import numpy as np

from .layout import Compressed


def random_compressed(geo, n_tracks: int, n_un: int, seed: int, max_ncl: int = 40, ncl=None, n_sectors_in: int = 36) -> Compressed:
    """Random bytes everywhere.  `ncl` (array) overrides the uniform 1..max_ncl track lengths."""
    rng = np.random.default_rng(seed)
    if ncl is None:
        ncl = rng.integers(1, max_ncl + 1, n_tracks).astype(np.uint16)
    else:
        ncl = np.asarray(ncl, np.uint16)
        n_tracks = len(ncl)
    n_att = int(ncl.astype(np.int64).sum())
    ucnt = rng.multinomial(n_un, np.full(geo.n_bins, 1.0 / geo.n_bins)).astype(np.uint32)
    c = Compressed.empty(n_tracks, n_att, n_un, geo.n_bins)
    c.trk_ncl[:] = ncl
    c.trk_qpt[:] = rng.integers(-128, 128, n_tracks)
    c.trk_row0[:] = rng.integers(0, geo.n_rows, n_tracks)
    c.trk_sec0[:] = rng.integers(0, n_sectors_in, n_tracks)
    c.trk_pad0[:] = rng.integers(0, 65536, n_tracks)
    c.trk_time0[:] = rng.integers(0, 2 ** 32, n_tracks)
    for k in ("a_qtot", "a_qmax", "a_padres", "u_qtot", "u_qmax", "u_paddiff"):
        getattr(c, k)[:] = rng.integers(0, 65536, len(getattr(c, k)))
    for k in ("a_flags", "a_sigpad", "a_sigtime", "a_rowdiff", "a_secleg", "u_flags", "u_sigpad", "u_sigtime"):
        getattr(c, k)[:] = rng.integers(0, 256, len(getattr(c, k)))
    for k in ("a_timeres", "u_timediff"):
        getattr(c, k)[:] = rng.integers(0, 2 ** 32, len(getattr(c, k)))
    c.u_bin_count[:] = ucnt
    return c


def degenerate_same_bin(geo, ncl, seed: int, n_un: int = 0) -> Compressed:
    """Every residual has rowdiff = 0 and no sector step: each track piles all its clusters into its first bin
    (stresses the rank / scatter with very long per-bin runs); half of the tracks share one start bin."""
    c = random_compressed(geo, 0, n_un, seed, ncl=ncl)
    c.a_rowdiff[:] = 0
    c.a_secleg[:] &= 0x80
    c.trk_row0[::2] = 7
    c.trk_sec0[::2] = 1
    return c
