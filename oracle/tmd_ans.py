"""Front end of the CPU oracle of the entropy stage (oracle/tmd_ans_oracle.c) and of the TMDZ container.  TEST INFRASTRUCTURE
ONLY: only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this module.

PAPER.md L20 ("lossless ANS"), L49 ("TPC Entropy Decoding"), L68 (track-model decoding starts "after the entropy decoding").
The container format is this build's own; it is restated here independently of the library's host encoder
and CUDA decoder (paper_2411_02206_b200/csrc/tmd_entropy*.{cuh,cu}), with which this module shares no code.

TMDZ, little endian:
  header (64 B): u32 magic 'TMDZ', u32 version 1, u32 n_tracks, u32 n_bins, u64 n_attached, u64 n_unattached,
                 u32 n_planes, u32 block_symbols (8192), u64 total_bytes, 16 B reserved
  plane directory, 32 B per plane: u32 array_id (index into the compressed SoA's 23 arrays), u32 byte_index, u64 n_symbols,
                 u64 table_offset (u16 freq[256], sums to 4096), u64 blocks_offset (u32 block_start[n_blocks + 1])
  A plane = byte `byte_index` of every element of an array (elements are 1, 2 or 4 bytes wide), coded in blocks of 8192
  symbols; block b occupies blob[block_start[b] : block_start[b + 1]] = 32 u32 coder states + the 16-bit words in decoder order.
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from tmd_inputs.layout import COMPRESSED_FIELDS, Compressed

from . import build as _build

MAGIC, VERSION, BLOCK, LANES = 0x5A444D54, 1, 8192, 32
HEADER_BYTES, PLANE_BYTES = 64, 32
_u8p, _u16p, _u32p = (C.POINTER(t) for t in (C.c_uint8, C.c_uint16, C.c_uint32))

_lib = None


def lib() -> C.CDLL:
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        _lib.orc_ans_build_table.restype = C.c_int
        _lib.orc_ans_encode_block.restype = C.c_int64
        _lib.orc_ans_decode_block.restype = C.c_int
    return _lib


def build_table(sym: np.ndarray) -> np.ndarray:
    sym = np.ascontiguousarray(sym, np.uint8)
    freq = np.zeros(256, np.uint16)
    rc = lib().orc_ans_build_table(sym.ctypes.data_as(_u8p), C.c_uint64(len(sym)), freq.ctypes.data_as(_u16p))
    if rc != 0:
        raise RuntimeError(f"orc_ans_build_table failed: {rc}")
    return freq


def encode_block(sym: np.ndarray, freq: np.ndarray) -> np.ndarray:
    sym = np.ascontiguousarray(sym, np.uint8)
    out = np.zeros(4 * LANES + 2 * len(sym) + 8, np.uint8)
    n = lib().orc_ans_encode_block(sym.ctypes.data_as(_u8p), C.c_uint32(len(sym)), freq.ctypes.data_as(_u16p),
                                   out.ctypes.data_as(_u8p), C.c_uint64(len(out)))
    if n < 0:
        raise RuntimeError(f"orc_ans_encode_block failed: {n}")
    return out[:n].copy()


def decode_block(data: np.ndarray, n: int, freq: np.ndarray, want_trace: bool = False):
    data = np.ascontiguousarray(data, np.uint8)
    sym = np.zeros(n, np.uint8)
    trace = np.zeros(n, np.uint32) if want_trace else None
    rc = lib().orc_ans_decode_block(data.ctypes.data_as(_u8p), C.c_uint64(len(data)), C.c_uint32(n), freq.ctypes.data_as(_u16p),
                                    sym.ctypes.data_as(_u8p), trace.ctypes.data_as(_u32p) if want_trace else None)
    if rc != 0:
        raise RuntimeError(f"orc_ans_decode_block failed: {rc}")
    return (sym, trace) if want_trace else sym


def planes_of(comp: Compressed):
    """(array_id, byte_index, symbols) for every byte plane of the compressed SoA, in container order."""
    for aid, (k, (dt, _)) in enumerate(COMPRESSED_FIELDS.items()):
        a = np.ascontiguousarray(getattr(comp, k))
        w = a.dtype.itemsize
        b = a.view(np.uint8).reshape(-1, w) if len(a) else np.zeros((0, w), np.uint8)
        for j in range(w):
            yield aid, j, np.ascontiguousarray(b[:, j])


def encode_container(comp: Compressed) -> np.ndarray:
    """Compressed SoA -> TMDZ blob (uint8 array)."""
    comp.check_shapes()
    planes = list(planes_of(comp))
    parts, directory = [], []
    pos = HEADER_BYTES + PLANE_BYTES * len(planes)

    def put(buf: np.ndarray, align: int = 16) -> int:
        nonlocal pos
        pad = (-pos) % align
        if pad:
            parts.append(np.zeros(pad, np.uint8)); pos += pad
        at = pos
        parts.append(np.ascontiguousarray(buf).view(np.uint8).reshape(-1)); pos += parts[-1].size
        return at

    for aid, j, sym in planes:
        freq = build_table(sym)
        t_off = put(freq)
        blocks = [encode_block(sym[i:i + BLOCK], freq) for i in range(0, len(sym), BLOCK)]
        starts = np.zeros(len(blocks) + 1, np.uint32)
        b_off = put(starts)                                  # placeholder, filled below
        slot = len(parts) - 1
        for i, blk in enumerate(blocks):
            starts[i] = put(blk, 4)
        starts[len(blocks)] = pos
        parts[slot] = starts.view(np.uint8)
        directory.append((aid, j, len(sym), t_off, b_off))
    total = pos
    head = np.zeros(HEADER_BYTES, np.uint8)
    head[:16].view(np.uint32)[:] = (MAGIC, VERSION, comp.n_tracks, comp.n_bins)
    head[16:32].view(np.uint64)[:] = (comp.n_attached, comp.n_unattached)
    head[32:40].view(np.uint32)[:] = (len(planes), BLOCK)
    head[40:48].view(np.uint64)[:] = (total,)
    d = np.zeros(PLANE_BYTES * len(planes), np.uint8)
    for i, (aid, j, n, t_off, b_off) in enumerate(directory):
        rec = d[PLANE_BYTES * i: PLANE_BYTES * (i + 1)]
        rec[:8].view(np.uint32)[:] = (aid, j)
        rec[8:32].view(np.uint64)[:] = (n, t_off, b_off)
    blob = np.concatenate([head, d] + parts)
    assert blob.size == total
    return blob


def decode_container(blob: np.ndarray) -> Compressed:
    """TMDZ blob -> compressed SoA (every plane decoded block by block with orc_ans_decode_block)."""
    blob = np.ascontiguousarray(blob, np.uint8)
    magic, version, n_trk, n_bins = blob[:16].view(np.uint32)
    n_att, n_un = (int(v) for v in blob[16:32].view(np.uint64))
    n_planes, block = (int(v) for v in blob[32:40].view(np.uint32))
    if magic != MAGIC or version != VERSION or block != BLOCK or int(blob[40:48].view(np.uint64)[0]) != blob.size:
        raise ValueError("not a TMDZ container")
    comp = Compressed.empty(int(n_trk), n_att, n_un, int(n_bins))
    names = list(COMPRESSED_FIELDS)
    for i in range(n_planes):
        rec = blob[HEADER_BYTES + PLANE_BYTES * i: HEADER_BYTES + PLANE_BYTES * (i + 1)]
        aid, j = (int(v) for v in rec[:8].view(np.uint32))
        n, t_off, b_off = (int(v) for v in rec[8:32].view(np.uint64))
        a = getattr(comp, names[aid])
        if n != len(a):
            raise ValueError(f"plane {i}: {n} symbols for {len(a)} elements")
        freq = blob[t_off:t_off + 512].view(np.uint16).copy()
        n_blocks = (n + BLOCK - 1) // BLOCK
        starts = blob[b_off:b_off + 4 * (n_blocks + 1)].view(np.uint32)
        out = a.view(np.uint8).reshape(-1, a.dtype.itemsize) if n else None
        for b in range(n_blocks):
            m = min(BLOCK, n - b * BLOCK)
            out[b * BLOCK: b * BLOCK + m, j] = decode_block(blob[int(starts[b]):int(starts[b + 1])], m, freq)
    return comp
