"""tmd_decode_unattached_noalloc: the entry point for callers that cannot allocate device memory.

Some users of libtmd run where cudaMalloc is off limits -- a framework grabbed the device's memory as one block at start-up,
or the code is a plug-in that only receives device pointers, or a latency-bound loop must not hit the device-wide
serialisation of cudaMalloc / cudaFree -- so they can neither call tmd_create (it allocates) nor bring a workspace.  For a
frame of unattached clusters the library therefore offers a call without context or workspace whose scratch is a fixed
64 KiB array inside the library image.  That array is shared by all calls on a device and keeps the last call's tables, so the
tests below call it several times in a row, with frames of different geometry and size, and demand each time exactly what the
ordinary path (tmd_create + tmd_decode with a caller-allocated workspace) writes: integer work, so the tolerance is zero --
byte-for-byte equality of the clusters and of bin_offset, as in every other GPU test of this repository.

This file is named to be collected last (`pytest --collect-only`): with `-x` a failure here must not hide other tests.  It
makes no assumption about what ran before it in the process and passes on its own in a fresh one.
"""
import numpy as np
import pytest

from tmd_inputs import build_geometry
from tmd_inputs.adversarial import random_compressed
from tmd_inputs.layout import CLUSTER_DTYPE, Compressed

from gpu_util import _as_torch, first_mismatch, gpu_decode

BZ = 0.5


def _unattached_frame(geo, counts, seed):
    """A frame without tracks whose bins hold `counts` unattached clusters; random bytes in every field."""
    rng = np.random.default_rng(seed)
    counts = np.asarray(counts, np.uint32)
    n = int(counts.sum())
    c = Compressed.empty(0, 0, n, geo.n_bins)
    c.u_bin_count[:] = counts
    c.u_paddiff[:] = rng.integers(0, 65536, n); c.u_timediff[:] = rng.integers(0, 2 ** 32, n)
    c.u_qtot[:] = rng.integers(0, 65536, n); c.u_qmax[:] = rng.integers(0, 65536, n)
    c.u_flags[:] = rng.integers(0, 256, n); c.u_sigpad[:] = rng.integers(0, 256, n); c.u_sigtime[:] = rng.integers(0, 256, n)
    return c


def _noalloc_decode(geo, comp, stream=None):
    """Run the no-allocation entry point on `comp` -> (clusters, bin_offset).  The test allocates inputs and outputs with torch,
    as any caller must; the library call itself gets no context and no workspace."""
    import torch
    from paper_2411_02206_b200 import tmd as T
    from tmd_inputs.layout import COMPRESSED_FIELDS

    n = comp.n_unattached
    dev = {k: _as_torch(np.ascontiguousarray(getattr(comp, k))).cuda() for k in COMPRESSED_FIELDS}
    d_clusters = torch.full((max(n, 1) * 16,), 0xEE, dtype=torch.uint8, device="cuda")
    d_binoff = torch.full((geo.n_bins + 1,), -1, dtype=torch.int32, device="cuda")
    c = T.make_compressed(dev)
    st = torch.cuda.current_stream() if stream is None else stream
    st.wait_stream(torch.cuda.current_stream())
    T.tmd_decode_unattached_noalloc(geo.n_sectors_out, geo.n_rows, c, d_clusters, d_binoff, st.cuda_stream)
    st.synchronize()
    clusters = d_clusters.cpu().numpy()[: n * 16].view(CLUSTER_DTYPE).copy()
    return clusters, d_binoff.cpu().numpy().view(np.uint32).copy()


def _assert_equals_existing_path(geo, comp, stream=None):
    want_cl, want_bo, _ = gpu_decode(geo, BZ, comp)                 # tmd_create + tmd_decode + caller workspace
    got_cl, got_bo = _noalloc_decode(geo, comp, stream)
    assert np.array_equal(got_bo, want_bo), "bin_offset: " + first_mismatch(got_bo, want_bo)
    assert got_cl.tobytes() == want_cl.tobytes(), "clusters: " + first_mismatch(got_cl.view(np.uint8), want_cl.view(np.uint8))


@pytest.mark.gpu
def test_two_calls_in_a_row_equal_the_workspace_path():
    """Back-to-back calls share the static scratch.  The second frame has FEWER bins (2 x 152 instead of 36 x 152) and other
    counts than the first, the third is the first geometry again with other counts: anything a call failed to rewrite --
    a stale start offset, a bin of the wider table -- would show up as a misplaced or missing cluster."""
    import torch
    geo36, geo2 = build_geometry(36), build_geometry(2)
    rng = np.random.default_rng(71)
    big = rng.poisson(30.0, geo36.n_bins)
    big[17] = 60_000                     # much larger than a tile: decoded by the whole block
    big[18] = 0
    big[19] = 1
    big[geo36.n_bins - 1] = 5000
    first = _unattached_frame(geo36, big, 72)
    second = _unattached_frame(geo2, rng.poisson(3.0, geo2.n_bins), 73)
    third = _unattached_frame(geo36, rng.poisson(700.0, geo36.n_bins), 74)      # >= 512 per bin: one block per bin
    _assert_equals_existing_path(geo36, first)
    _assert_equals_existing_path(geo2, second)
    _assert_equals_existing_path(geo36, third)
    _assert_equals_existing_path(geo36, first, stream=torch.cuda.Stream())      # and once more, on a stream of the caller's


@pytest.mark.gpu
def test_empty_frames_and_the_same_frame_twice():
    geo = build_geometry(36)
    empty = Compressed.empty(0, 0, 0, geo.n_bins)
    cl, bo = _noalloc_decode(geo, empty)
    assert len(cl) == 0 and np.all(bo == 0)
    frame = random_compressed(geo, 0, 40_000, 75)
    a = _noalloc_decode(geo, frame)
    b = _noalloc_decode(geo, frame)
    assert a[0].tobytes() == b[0].tobytes() and np.array_equal(a[1], b[1])
    _assert_equals_existing_path(geo, frame)


def test_sizes_beyond_the_static_scratch_are_refused():
    """Pure argument checks: they come before any CUDA call, so this runs without a GPU."""
    import ctypes as C
    from paper_2411_02206_b200 import tmd as T
    L = T.lib()
    c = T.tmd_compressed(0, 0, 0)
    c.u_bin_count = 0x1000                     # never dereferenced: the call is refused first
    assert T.TMD_NOALLOC_MAX_BINS == 8192
    # 54 x 152 = 8208 bins > 8192: would not fit the built-in tables
    assert L.tmd_decode_unattached_noalloc(54, 152, C.byref(c), None, 0x1000, None) == T.TMD_ERR_LIMIT
    assert L.tmd_decode_unattached_noalloc(126, 255, C.byref(c), None, 0x1000, None) == T.TMD_ERR_LIMIT
    big = T.tmd_compressed(0, 0, 0xFFFF0001)
    big.u_bin_count = 0x1000
    assert L.tmd_decode_unattached_noalloc(36, 152, C.byref(big), 0x1000, 0x1000, None) == T.TMD_ERR_LIMIT
    # frames with tracks belong to tmd_decode
    trk = T.tmd_compressed(1, 1, 0)
    trk.u_bin_count = 0x1000
    assert L.tmd_decode_unattached_noalloc(36, 152, C.byref(trk), None, 0x1000, None) == T.TMD_ERR_ARG
    assert L.tmd_decode_unattached_noalloc(36, 152, None, None, 0x1000, None) == T.TMD_ERR_ARG
    assert L.tmd_decode_unattached_noalloc(36, 152, C.byref(c), None, None, None) == T.TMD_ERR_ARG
    assert L.tmd_decode_unattached_noalloc(36, 256, C.byref(c), None, 0x1000, None) == T.TMD_ERR_ARG
    assert "built-in scratch" in T.tmd_status_string(T.TMD_ERR_LIMIT)
