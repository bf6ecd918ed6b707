"""ctypes front end of the CPU oracle (oracle/tmd_oracle.c).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this module.
It never imports the CUDA package.  Paper passages followed: PAPER.md L68, L70 (see the C file's header).
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from tmd_inputs.geometry import Geometry
from tmd_inputs.layout import CLUSTER_DTYPE, COMPRESSED_FIELDS, Compressed

from . import build as _build

_u8p, _i8p, _u16p, _u32p, _f32p = (C.POINTER(t) for t in (C.c_uint8, C.c_int8, C.c_uint16, C.c_uint32, C.c_float))
_CT = {"<u2": _u16p, "i1": _i8p, "u1": _u8p, "<u4": _u32p}


class _Geometry(C.Structure):
    _fields_ = [("n_az", C.c_uint32), ("n_sides", C.c_uint32), ("n_sectors_out", C.c_uint32), ("n_rows", C.c_uint32),
                ("cos_a", C.c_float), ("sin_a", C.c_float), ("bz_tesla", C.c_float),
                ("row_x", _f32p), ("row_padw", _f32p), ("row_inv_padw", _f32p), ("row_npads", _u16p)]


class _Compressed(C.Structure):
    _fields_ = [("n_tracks", C.c_uint32), ("n_attached", C.c_uint64), ("n_unattached", C.c_uint64)] + \
               [(k, _CT[dt]) for k, (dt, _) in COMPRESSED_FIELDS.items()]


class TraceRow(C.Structure):
    _fields_ = [("sec", C.c_uint32), ("row", C.c_uint32), ("dir", C.c_int32), ("ok", C.c_int32)] + \
               [(k, C.c_uint32) for k in ("x", "y", "sp", "sp2", "y2", "u2", "s", "P_pred", "T_pred", "P", "T",
                                          "yn", "un", "spn", "dtn", "kn")]


_lib = None


def lib() -> C.CDLL:
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        _lib.orc_decode.restype = C.c_int
        _lib.orc_decode_track.restype = C.c_int
        _lib.orc_encode.restype = C.c_int
    return _lib


def _ptr(a: np.ndarray, typ):
    assert a.flags["C_CONTIGUOUS"]
    return a.ctypes.data_as(typ)


def _geom(g: Geometry, bz_tesla: float):
    keep = [np.ascontiguousarray(g.row_x, np.float32), np.ascontiguousarray(g.row_padw, np.float32),
            np.ascontiguousarray(g.row_inv_padw, np.float32), np.ascontiguousarray(g.row_npads, np.uint16)]
    s = _Geometry(g.n_az, g.n_sides, g.n_sectors_out, g.n_rows, float(g.cos_a), float(g.sin_a), float(np.float32(bz_tesla)),
                  _ptr(keep[0], _f32p), _ptr(keep[1], _f32p), _ptr(keep[2], _f32p), _ptr(keep[3], _u16p))
    return s, keep


def _comp(c: Compressed):
    c.check_shapes()
    s = _Compressed(c.n_tracks, c.n_attached, c.n_unattached)
    keep = []
    for k, (dt, _) in COMPRESSED_FIELDS.items():
        a = np.ascontiguousarray(getattr(c, k))
        keep.append(a)
        setattr(s, k, _ptr(a, _CT[dt]))
    return s, keep


def decode(g: Geometry, bz_tesla: float, c: Compressed, probe_step: int | None = None):
    """Full decode -> (clusters[CLUSTER_DTYPE], bin_offset u32[n_bins+1], probe bits u32[n_tracks,6] or None)."""
    gs, k1 = _geom(g, bz_tesla)
    cs, k2 = _comp(c)
    n = c.n_attached + c.n_unattached
    clusters = np.zeros(n, dtype=CLUSTER_DTYPE)
    bin_offset = np.zeros(g.n_bins + 1, dtype=np.uint32)
    probes = np.zeros((c.n_tracks, 6), dtype=np.uint32) if probe_step is not None else None
    rc = lib().orc_decode(C.byref(gs), C.byref(cs), C.c_void_p(clusters.ctypes.data), _ptr(bin_offset, _u32p),
                          _ptr(probes, _u32p) if probes is not None else None,
                          C.c_uint32(0xFFFFFFFF if probe_step is None else probe_step))
    if rc != 0:
        raise RuntimeError(f"orc_decode failed: {rc}")
    return clusters, bin_offset, probes


def decode_track(g: Geometry, bz_tesla: float, qpt: int, sec0: int, row0: int, P0: int, T0: int,
                 rowdiff, secleg, padres, timeres, want_trace: bool = False, probe_step: int | None = None):
    """Decode one track -> dict(sec,row,P,T[, trace rows][, probe])."""
    gs, k1 = _geom(g, bz_tesla)
    rowdiff = np.ascontiguousarray(rowdiff, np.uint8)
    secleg = np.ascontiguousarray(secleg, np.uint8)
    padres = np.ascontiguousarray(np.asarray(padres, dtype=np.int64) & 0xFFFF, np.uint16)
    timeres = np.ascontiguousarray(np.asarray(timeres, dtype=np.int64) & 0xFFFFFFFF, np.uint32)
    ncl = len(rowdiff) + 1
    sec = np.zeros(ncl, np.uint8); row = np.zeros(ncl, np.uint8)
    P = np.zeros(ncl, np.uint16); T = np.zeros(ncl, np.uint32)
    trace = (TraceRow * max(ncl - 1, 1))() if want_trace else None
    probe = np.zeros(6, np.uint32) if probe_step is not None else None
    rc = lib().orc_decode_track(C.byref(gs), C.c_int8(qpt), C.c_uint32(sec0), C.c_uint32(row0), C.c_uint32(P0), C.c_uint32(T0),
                                C.c_uint32(ncl), _ptr(rowdiff, _u8p), _ptr(secleg, _u8p), _ptr(padres, _u16p),
                                _ptr(timeres, _u32p), _ptr(sec, _u8p), _ptr(row, _u8p), _ptr(P, _u16p), _ptr(T, _u32p),
                                trace, C.c_uint32(0xFFFFFFFF if probe_step is None else probe_step),
                                _ptr(probe, _u32p) if probe is not None else None)
    if rc != 0:
        raise RuntimeError(f"orc_decode_track failed: {rc}")
    out = {"sec": sec, "row": row, "P": P, "T": T}
    if want_trace:
        out["trace"] = [trace[i] for i in range(ncl - 1)]
    if probe is not None:
        out["probe"] = probe
    return out


def encode(g: Geometry, bz_tesla: float, trk_ncl, trk_qptf, att: np.ndarray, leg, un: np.ndarray) -> Compressed:
    """Oracle encoder: g-ordered attached clusters + unattached clusters -> Compressed."""
    gs, k1 = _geom(g, bz_tesla)
    trk_ncl = np.ascontiguousarray(trk_ncl, np.uint16)
    trk_qptf = np.ascontiguousarray(trk_qptf, np.float32)
    att = np.ascontiguousarray(att, CLUSTER_DTYPE)
    un = np.ascontiguousarray(un, CLUSTER_DTYPE)
    leg = np.ascontiguousarray(leg, np.uint8)
    n_trk, n_att, n_un = len(trk_ncl), len(att), len(un)
    assert len(leg) == n_att and len(trk_qptf) == n_trk
    out = Compressed.empty(n_trk, n_att, n_un, g.n_bins)
    out.trk_ncl[:] = trk_ncl
    order = ["trk_qpt", "trk_row0", "trk_sec0", "trk_pad0", "trk_time0",
             "a_qtot", "a_qmax", "a_flags", "a_sigpad", "a_sigtime",
             "a_rowdiff", "a_secleg", "a_padres", "a_timeres",
             "u_qtot", "u_qmax", "u_flags", "u_sigpad", "u_sigtime", "u_paddiff", "u_timediff", "u_bin_count"]
    args = [_ptr(getattr(out, k), _CT[COMPRESSED_FIELDS[k][0]]) for k in order]
    rc = lib().orc_encode(C.byref(gs), C.c_uint32(n_trk), _ptr(trk_ncl, _u16p), _ptr(trk_qptf, _f32p),
                          C.c_uint64(n_att), C.c_void_p(att.ctypes.data), _ptr(leg, _u8p),
                          C.c_uint64(n_un), C.c_void_p(un.ctypes.data), *args)
    if rc != 0:
        raise RuntimeError(f"orc_encode failed: {rc}")
    return out
