"""ctypes binding of libtmd.so -- same names as include/tmd.h, argument marshalling only.

Every step of the path (offsets scan, geometry walk + ranks, column scan, track-model decode, scatter, unattached
prefix sums) runs in the CUDA kernels of csrc/.  PyTorch supplies device memory and streams, nothing else.
PAPER.md L68/L70 define the operation; include/tmd.h states layout, ownership and error behaviour.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

_HERE = os.path.dirname(os.path.abspath(__file__))

TMD_OK, TMD_ERR_ARG, TMD_ERR_ALIGN, TMD_ERR_WORKSPACE, TMD_ERR_CUDA, TMD_ERR_CORRUPT, TMD_ERR_DEVICE, TMD_ERR_LIMIT = 0, -1, -2, -3, -4, -5, -6, -7
TMD_NOALLOC_MAX_BINS = 8192
TMD_VALIDATE = 1
TMD_TIMING = 2
TMD_MAX_KERNELS = 24
TMD_MAX_BATCH = 1024
TMD_HOST_SLOTS = 2
PROBE_FINAL = 0xFFFFFFFF

# (field name, numpy dtype) in the order of struct tmd_compressed
COMPRESSED_ARRAYS = (
    ("trk_ncl", "<u2"), ("trk_qpt", "i1"), ("trk_row0", "u1"), ("trk_sec0", "u1"), ("trk_pad0", "<u2"), ("trk_time0", "<u4"),
    ("a_qtot", "<u2"), ("a_qmax", "<u2"), ("a_flags", "u1"), ("a_sigpad", "u1"), ("a_sigtime", "u1"),
    ("a_rowdiff", "u1"), ("a_secleg", "u1"), ("a_padres", "<u2"), ("a_timeres", "<u4"),
    ("u_qtot", "<u2"), ("u_qmax", "<u2"), ("u_flags", "u1"), ("u_sigpad", "u1"), ("u_sigtime", "u1"),
    ("u_paddiff", "<u2"), ("u_timediff", "<u4"), ("u_bin_count", "<u4"),
)


class tmd_geometry(C.Structure):
    _fields_ = [("n_az", C.c_uint32), ("n_sides", C.c_uint32), ("n_sectors_out", C.c_uint32), ("n_rows", C.c_uint32),
                ("cos_a", C.c_float), ("sin_a", C.c_float),
                ("row_x", C.c_void_p), ("row_padw", C.c_void_p), ("row_inv_padw", C.c_void_p), ("row_npads", C.c_void_p)]


class tmd_field(C.Structure):
    _fields_ = [("bz_tesla", C.c_float)]


class tmd_compressed(C.Structure):
    _fields_ = [("n_tracks", C.c_uint32), ("n_attached", C.c_uint64), ("n_unattached", C.c_uint64)] + \
               [(k, C.c_void_p) for k, _ in COMPRESSED_ARRAYS]


class tmd_output(C.Structure):
    _fields_ = [("clusters", C.c_void_p), ("bin_offset", C.c_void_p), ("probe_state", C.c_void_p),
                ("probe_step", C.c_uint32), ("workspace", C.c_void_p), ("workspace_bytes", C.c_size_t)]


class tmd_attached_truth(C.Structure):
    _fields_ = [("n_tracks", C.c_uint32), ("n_attached", C.c_uint64), ("trk_ncl", C.c_void_p), ("trk_qptf", C.c_void_p),
                ("att", C.c_void_p), ("leg", C.c_void_p)]


_lib = None


def lib() -> C.CDLL:
    """Load (building first if the sources are newer) libtmd.so.  Raises if that is impossible: no fallback."""
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(path)
        L.tmd_create.argtypes = [C.POINTER(tmd_geometry), C.POINTER(tmd_field), C.POINTER(C.c_void_p)]
        L.tmd_workspace_bytes.argtypes = [C.c_void_p, C.c_uint32, C.c_uint64, C.c_uint64, C.POINTER(C.c_size_t)]
        L.tmd_decode.argtypes = [C.c_void_p, C.POINTER(tmd_compressed), C.POINTER(tmd_output), C.c_uint32, C.c_void_p]
        L.tmd_decode_host.argtypes = L.tmd_decode.argtypes
        L.tmd_decode_batch.argtypes = [C.c_void_p, C.c_uint32, C.POINTER(tmd_compressed), C.POINTER(tmd_output), C.c_uint32, C.c_void_p]
        L.tmd_decode_batch.restype = C.c_int
        L.tmd_destroy.argtypes = [C.c_void_p]
        L.tmd_status_string.argtypes = [C.c_int]
        L.tmd_status_string.restype = C.c_char_p
        L.tmd_last_launch_count.argtypes = [C.c_void_p]
        L.tmd_kernel_times.argtypes = [C.c_void_p, C.c_int, C.POINTER(C.c_char_p), C.POINTER(C.c_float)]
        L.tmd_encode_attached.argtypes = [C.c_void_p, C.POINTER(tmd_attached_truth), C.POINTER(tmd_compressed), C.c_void_p,
                                          C.c_size_t, C.c_void_p]
        L.tmd_decode_host_async.argtypes = [C.c_void_p, C.POINTER(tmd_compressed), C.POINTER(tmd_output), C.c_uint32, C.c_int]
        L.tmd_host_wait.argtypes = [C.c_void_p, C.c_int]
        L.tmd_decode_container_host_async.argtypes = [C.c_void_p, C.c_void_p, C.c_size_t, C.POINTER(tmd_output), C.c_uint32, C.c_int]
        L.tmd_decode_container_host_async.restype = C.c_int
        L.tmd_encode_unattached_workspace_bytes.argtypes = [C.c_void_p, C.c_uint64, C.POINTER(C.c_size_t)]
        L.tmd_encode_unattached_workspace_bytes.restype = C.c_int
        L.tmd_encode_unattached.argtypes = [C.c_void_p, C.c_uint64, C.c_void_p, C.POINTER(tmd_compressed), C.c_void_p, C.c_size_t, C.c_void_p]
        L.tmd_encode_unattached.restype = C.c_int
        L.tmd_entropy_bound.argtypes = [C.c_uint32, C.c_uint64, C.c_uint64, C.c_uint32, C.POINTER(C.c_size_t)]
        L.tmd_entropy_encode_host.argtypes = [C.POINTER(tmd_compressed), C.c_uint32, C.c_void_p, C.c_size_t, C.POINTER(C.c_size_t)]
        L.tmd_entropy_sizes.argtypes = [C.c_void_p, C.c_size_t, C.POINTER(C.c_uint32), C.POINTER(C.c_uint64), C.POINTER(C.c_uint64), C.POINTER(C.c_uint32), C.POINTER(C.c_size_t)]
        L.tmd_entropy_decode.argtypes = [C.c_void_p, C.c_size_t, C.c_void_p, C.c_size_t, C.POINTER(tmd_compressed), C.c_void_p, C.c_void_p]
        for f in (L.tmd_entropy_bound, L.tmd_entropy_encode_host, L.tmd_entropy_sizes, L.tmd_entropy_decode):
            f.restype = C.c_int
        L.tmd_decode_unattached_noalloc.argtypes = [C.c_uint32, C.c_uint32, C.POINTER(tmd_compressed), C.c_void_p, C.c_void_p, C.c_void_p]
        L.tmd_decode_unattached_noalloc.restype = C.c_int
        L.tmd_selftest_ieee.argtypes = [C.c_uint32, C.POINTER(C.c_uint64)]
        L.tmd_selftest_ieee.restype = C.c_int
        L.tmd_decode_host_async.restype = C.c_int
        L.tmd_host_wait.restype = C.c_int
        L.tmd_kernel_times.restype = C.c_int
        L.tmd_encode_attached.restype = C.c_int
        for f in (L.tmd_create, L.tmd_workspace_bytes, L.tmd_decode, L.tmd_decode_host, L.tmd_destroy, L.tmd_last_launch_count):
            f.restype = C.c_int
        _lib = L
    return _lib


class TmdError(RuntimeError):
    def __init__(self, status: int):
        self.status = status
        super().__init__(f"tmd status {status}: {tmd_status_string(status)}")


def tmd_status_string(status: int) -> str:
    return lib().tmd_status_string(status).decode()


def _check(rc: int) -> None:
    if rc != TMD_OK:
        raise TmdError(rc)


def _ptr(a) -> int | None:
    """Address of a torch tensor (device or host) or numpy array; None for absent / empty arrays."""
    if a is None:
        return None
    if isinstance(a, np.ndarray):
        assert a.flags["C_CONTIGUOUS"]
        return a.ctypes.data if a.size else None
    assert a.is_contiguous()
    return a.data_ptr() if a.numel() else None


def tmd_create(geo, bz_tesla: float) -> int:
    """tmd_create(geometry, field) -> opaque context handle.  `geo` = tmd_inputs.geometry.Geometry (tables as inputs)."""
    keep = [np.ascontiguousarray(geo.row_x, np.float32), np.ascontiguousarray(geo.row_padw, np.float32),
            np.ascontiguousarray(geo.row_inv_padw, np.float32), np.ascontiguousarray(geo.row_npads, np.uint16)]
    g = tmd_geometry(geo.n_az, geo.n_sides, geo.n_sectors_out, geo.n_rows, float(geo.cos_a), float(geo.sin_a),
                     *(k.ctypes.data for k in keep))
    f = tmd_field(float(np.float32(bz_tesla)))
    ctx = C.c_void_p()
    _check(lib().tmd_create(C.byref(g), C.byref(f), C.byref(ctx)))
    return ctx.value


def tmd_destroy(ctx: int) -> None:
    _check(lib().tmd_destroy(ctx))


def tmd_workspace_bytes(ctx: int, n_tracks: int, n_attached: int, n_unattached: int) -> int:
    out = C.c_size_t()
    _check(lib().tmd_workspace_bytes(ctx, n_tracks, n_attached, n_unattached, C.byref(out)))
    return out.value


def tmd_last_launch_count(ctx: int) -> int:
    return lib().tmd_last_launch_count(ctx)


def make_compressed(arrays: dict) -> tmd_compressed:
    """struct tmd_compressed from a dict name -> tensor/ndarray (all on the device, or all on the host)."""
    n_trk = int(arrays["trk_ncl"].shape[0])
    n_att = int(arrays["a_qtot"].shape[0])
    n_un = int(arrays["u_qtot"].shape[0])
    c = tmd_compressed(n_trk, n_att, n_un)
    for k, _ in COMPRESSED_ARRAYS:
        setattr(c, k, _ptr(arrays[k]))
    return c


def make_output(clusters, bin_offset, workspace=None, probe_state=None, probe_step: int = PROBE_FINAL) -> tmd_output:
    ws_bytes = 0 if workspace is None else int(workspace.numel() * workspace.element_size())
    return tmd_output(_ptr(clusters), _ptr(bin_offset), _ptr(probe_state), probe_step, _ptr(workspace), ws_bytes)


def tmd_decode(ctx: int, comp: tmd_compressed, out: tmd_output, flags: int = 0, stream: int = 0) -> None:
    """Enqueue the decode of one time frame on CUDA stream handle `stream` (DEVICE pointers)."""
    _check(lib().tmd_decode(ctx, C.byref(comp), C.byref(out), flags, stream))


def make_batch(comps: list, outs: list):
    """(n_frames, tmd_compressed[n], tmd_output[n]) as contiguous HOST arrays of the structs, for tmd_decode_batch."""
    assert len(comps) == len(outs) and len(comps) >= 1
    n = len(comps)
    ca, oa = (tmd_compressed * n)(*comps), (tmd_output * n)(*outs)
    return n, ca, oa


def tmd_decode_batch(ctx: int, batch, flags: int = 0, stream: int = 0) -> None:
    """Enqueue the decode of all frames of `batch` (from make_batch) with one launch sequence on CUDA stream `stream`."""
    n, ca, oa = batch
    _check(lib().tmd_decode_batch(ctx, n, ca, oa, flags, stream))


def tmd_decode_host(ctx: int, comp: tmd_compressed, out: tmd_output, flags: int = 0, stream: int = 0) -> None:
    """End-to-end decode with HOST pointers (copies in, decodes, copies out, synchronises)."""
    _check(lib().tmd_decode_host(ctx, C.byref(comp), C.byref(out), flags, stream))


def tmd_decode_host_async(ctx: int, comp: tmd_compressed, out: tmd_output, flags: int = 0, slot: int = 0) -> None:
    """Enqueue upload + decode + download of one time frame (pinned HOST pointers) in pipeline slot `slot`; returns at once."""
    _check(lib().tmd_decode_host_async(ctx, C.byref(comp), C.byref(out), flags, slot))


def tmd_decode_container_host_async(ctx: int, blob, out: tmd_output, flags: int = 0, slot: int = 0) -> None:
    """Enqueue upload of a TMDZ container (HOST uint8 array / pinned tensor) + entropy decode + track-model decode + download of
    the clusters in pipeline slot `slot`; returns at once.  tmd_host_wait(slot) raises TMD_ERR_CORRUPT for a damaged container."""
    n = int(blob.size if isinstance(blob, np.ndarray) else blob.numel())
    _check(lib().tmd_decode_container_host_async(ctx, _ptr(blob), n, C.byref(out), flags, slot))


def tmd_host_wait(ctx: int, slot: int = 0) -> None:
    """Block until the frame in pipeline slot `slot` is complete in its host buffers."""
    _check(lib().tmd_host_wait(ctx, slot))


def tmd_decode_unattached_noalloc(n_sectors_out: int, n_rows: int, comp: tmd_compressed, clusters, bin_offset, stream: int = 0) -> None:
    """Enqueue the decode of a frame that holds only unattached clusters, for callers that cannot allocate device memory
    (no context, no workspace: the scratch is a fixed array inside libtmd.so; at most TMD_NOALLOC_MAX_BINS bins, else
    TmdError(TMD_ERR_LIMIT)).  `comp.u_*`, `clusters`, `bin_offset`: DEVICE memory.  Calls on one device share the scratch:
    keep them ordered (one stream, or events); see include/tmd.h."""
    _check(lib().tmd_decode_unattached_noalloc(n_sectors_out, n_rows, C.byref(comp), _ptr(clusters), _ptr(bin_offset), stream))


def tmd_selftest_ieee(log2_pairs: int = 32) -> tuple[int, int, int]:
    """Mismatch counts (sqrt, div, floor-clamp) of the kernel's unchecked IEEE sequences against the intrinsics; all 0."""
    m = (C.c_uint64 * 3)()
    _check(lib().tmd_selftest_ieee(log2_pairs, m))
    return int(m[0]), int(m[1]), int(m[2])


def tmd_kernel_times(ctx: int) -> list[tuple[str, float]]:
    """(kernel name, milliseconds) of the last tmd_decode that ran with TMD_TIMING, in launch order."""
    names = (C.c_char_p * TMD_MAX_KERNELS)()
    ms = (C.c_float * TMD_MAX_KERNELS)()
    n = lib().tmd_kernel_times(ctx, TMD_MAX_KERNELS, names, ms)
    if n < 0:
        raise TmdError(n)
    return [(names[i].decode(), float(ms[i])) for i in range(n)]


def tmd_encode_attached(ctx: int, trk_ncl, trk_qptf, att, leg, out_arrays: dict, workspace, stream: int = 0) -> None:
    """Encode g-ordered attached clusters (DEVICE tensors) into the trk_* / a_* arrays of `out_arrays` (DEVICE, writable)."""
    truth = tmd_attached_truth(int(trk_ncl.shape[0]), int(leg.shape[0]), _ptr(trk_ncl), _ptr(trk_qptf), _ptr(att), _ptr(leg))
    c = tmd_compressed(truth.n_tracks, truth.n_attached, 0)
    for k, _ in COMPRESSED_ARRAYS:
        if k in out_arrays:
            setattr(c, k, _ptr(out_arrays[k]))
    ws_bytes = int(workspace.numel() * workspace.element_size())
    _check(lib().tmd_encode_attached(ctx, C.byref(truth), C.byref(c), _ptr(workspace), ws_bytes, stream))


def tmd_encode_unattached_workspace_bytes(ctx: int, n_unattached: int) -> int:
    out = C.c_size_t()
    _check(lib().tmd_encode_unattached_workspace_bytes(ctx, n_unattached, C.byref(out)))
    return out.value


def tmd_encode_unattached(ctx: int, un, out_arrays: dict, workspace, stream: int = 0) -> None:
    """Encode unattached clusters (DEVICE tensor of 16-byte records, any order) into the u_* arrays and u_bin_count of
    `out_arrays` (DEVICE, writable)."""
    n = int(un.shape[0])
    c = tmd_compressed(0, 0, n)
    for k, _ in COMPRESSED_ARRAYS:
        if k in out_arrays:
            setattr(c, k, _ptr(out_arrays[k]))
    ws_bytes = int(workspace.numel() * workspace.element_size())
    _check(lib().tmd_encode_unattached(ctx, n, _ptr(un), C.byref(c), _ptr(workspace), ws_bytes, stream))


ENTROPY_HEAD_BYTES = 64 + 32 * 43


def tmd_entropy_bound(n_tracks: int, n_attached: int, n_unattached: int, n_bins: int) -> int:
    out = C.c_size_t()
    _check(lib().tmd_entropy_bound(n_tracks, n_attached, n_unattached, n_bins, C.byref(out)))
    return out.value


def tmd_entropy_encode_host(host_arrays: dict, n_bins: int) -> np.ndarray:
    """Compressed SoA (HOST numpy arrays / CPU tensors) -> TMDZ container (numpy uint8 array), encoded on the host."""
    comp = make_compressed(host_arrays)
    cap = tmd_entropy_bound(comp.n_tracks, comp.n_attached, comp.n_unattached, n_bins)
    blob = np.empty(cap, np.uint8)
    n = C.c_size_t()
    _check(lib().tmd_entropy_encode_host(C.byref(comp), n_bins, blob.ctypes.data, cap, C.byref(n)))
    return blob[: n.value].copy()


def tmd_entropy_sizes(head: np.ndarray) -> tuple[int, int, int, int, int]:
    """(n_tracks, n_attached, n_unattached, n_bins, container bytes) from a container's first bytes (HOST)."""
    a, b, c, d, e = C.c_uint32(), C.c_uint64(), C.c_uint64(), C.c_uint32(), C.c_size_t()
    _check(lib().tmd_entropy_sizes(head.ctypes.data, head.size, C.byref(a), C.byref(b), C.byref(c), C.byref(d), C.byref(e)))
    return a.value, b.value, c.value, d.value, e.value


def tmd_entropy_decode(head: np.ndarray, d_blob, out_arrays: dict, d_err, stream: int = 0) -> None:
    """Enqueue the decode of the TMDZ container `d_blob` (DEVICE uint8 tensor) into the DEVICE arrays of `out_arrays`."""
    comp = make_compressed(out_arrays)
    _check(lib().tmd_entropy_decode(head.ctypes.data, head.size, _ptr(d_blob), int(d_blob.numel()), C.byref(comp), _ptr(d_err), stream))
