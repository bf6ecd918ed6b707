"""Data layout of the track-model decoder's input and output (no arithmetic).

Input  = the "input Structure Of Arrays (SOA)" the paper names (§4) after entropy
         decoding; array names/widths are SURVEY.md §8(c)-C2.
Output = 16-byte cluster records in canonical per-(sector,row) order.
"""
from __future__ import annotations

from dataclasses import dataclass, fields

import numpy as np

N_AZ = 18       # azimuthal sectors per side
N_SIDES = 2     # A, C
N_ROWS = 152    # pad rows per sector

# u32 time; u16 pad; u16 qtot; u16 qmax; u8 sigpad; u8 sigtime; u8 flags; u8 row; u8 sector; u8 zero
CLUSTER_DTYPE = np.dtype(
    [("time", "<u4"), ("pad", "<u2"), ("qtot", "<u2"), ("qmax", "<u2"),
     ("sigpad", "u1"), ("sigtime", "u1"), ("flags", "u1"),
     ("row", "u1"), ("sector", "u1"), ("zero", "u1")]
)
assert CLUSTER_DTYPE.itemsize == 16

# name -> (dtype, which length it has)
COMPRESSED_FIELDS = {
    # per track
    "trk_ncl": ("<u2", "n_tracks"), "trk_qpt": ("i1", "n_tracks"),
    "trk_row0": ("u1", "n_tracks"), "trk_sec0": ("u1", "n_tracks"),
    "trk_pad0": ("<u2", "n_tracks"), "trk_time0": ("<u4", "n_tracks"),
    # per attached cluster (incl. each track's first), index g = off[t] + j
    "a_qtot": ("<u2", "n_attached"), "a_qmax": ("<u2", "n_attached"), "a_flags": ("u1", "n_attached"),
    "a_sigpad": ("u1", "n_attached"), "a_sigtime": ("u1", "n_attached"),
    # per attached cluster excluding each track's first, index g - t - 1
    "a_rowdiff": ("u1", "n_residuals"), "a_secleg": ("u1", "n_residuals"),
    "a_padres": ("<u2", "n_residuals"), "a_timeres": ("<u4", "n_residuals"),
    # per unattached cluster, bin after bin
    "u_qtot": ("<u2", "n_unattached"), "u_qmax": ("<u2", "n_unattached"), "u_flags": ("u1", "n_unattached"),
    "u_sigpad": ("u1", "n_unattached"), "u_sigtime": ("u1", "n_unattached"),
    "u_paddiff": ("<u2", "n_unattached"), "u_timediff": ("<u4", "n_unattached"),
    # per output bin (sector * n_rows + row)
    "u_bin_count": ("<u4", "n_bins"),
}


@dataclass
class Compressed:
    """Compressed-cluster SoA of one time frame as host numpy arrays."""
    trk_ncl: np.ndarray
    trk_qpt: np.ndarray
    trk_row0: np.ndarray
    trk_sec0: np.ndarray
    trk_pad0: np.ndarray
    trk_time0: np.ndarray
    a_qtot: np.ndarray
    a_qmax: np.ndarray
    a_flags: np.ndarray
    a_sigpad: np.ndarray
    a_sigtime: np.ndarray
    a_rowdiff: np.ndarray
    a_secleg: np.ndarray
    a_padres: np.ndarray
    a_timeres: np.ndarray
    u_qtot: np.ndarray
    u_qmax: np.ndarray
    u_flags: np.ndarray
    u_sigpad: np.ndarray
    u_sigtime: np.ndarray
    u_paddiff: np.ndarray
    u_timediff: np.ndarray
    u_bin_count: np.ndarray

    @property
    def n_tracks(self) -> int:
        return int(self.trk_ncl.shape[0])

    @property
    def n_attached(self) -> int:
        return int(self.a_qtot.shape[0])

    @property
    def n_residuals(self) -> int:
        return int(self.a_rowdiff.shape[0])

    @property
    def n_unattached(self) -> int:
        return int(self.u_qtot.shape[0])

    @property
    def n_bins(self) -> int:
        return int(self.u_bin_count.shape[0])

    def check_shapes(self) -> None:
        """Array lengths and dtypes agree with COMPRESSED_FIELDS (no value checks)."""
        lens = {"n_tracks": self.n_tracks, "n_attached": self.n_attached,
                "n_residuals": self.n_attached - self.n_tracks,
                "n_unattached": self.n_unattached, "n_bins": self.n_bins}
        for f in fields(self):
            a = getattr(self, f.name)
            dt, which = COMPRESSED_FIELDS[f.name]
            if a.dtype != np.dtype(dt) or a.ndim != 1 or a.shape[0] != lens[which]:
                raise ValueError(f"{f.name}: got {a.dtype}{a.shape}, want {dt}[{lens[which]}]")

    def nbytes(self) -> int:
        return sum(getattr(self, f.name).nbytes for f in fields(self))

    @staticmethod
    def empty(n_tracks: int, n_attached: int, n_unattached: int, n_bins: int) -> "Compressed":
        lens = {"n_tracks": n_tracks, "n_attached": n_attached, "n_residuals": n_attached - n_tracks,
                "n_unattached": n_unattached, "n_bins": n_bins}
        return Compressed(**{k: np.zeros(lens[w], dtype=dt) for k, (dt, w) in COMPRESSED_FIELDS.items()})


def algorithmic_bytes(n_tracks: int, n_attached: int, n_unattached: int, n_bins: int) -> int:
    """Bytes the method must move: compressed SoA in + 16-B records and bin offsets out."""
    b_in = 11 * n_tracks + 7 * n_attached + 8 * (n_attached - n_tracks) + 13 * n_unattached + 4 * n_bins
    b_out = 16 * (n_attached + n_unattached) + 4 * (n_bins + 1)
    return b_in + b_out
