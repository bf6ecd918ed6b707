"""`-m gpu` parity at BASELINE.json's full sizes, in the launch configuration bench.py times (same workload builder, same
`tmd_decode` call: flags 0, no probes, workspace from `tmd_workspace_bytes`).

A full time frame (c3: 251 M attached + 80 M unattached clusters) is more than the oracle decodes in seconds, so:

1. EVERY output record is compared, on the device with torch library routines only, against what the method's definition
   fixes at any size -- `decode(encode(x)) == canonical(x)` (pinned for the oracle at small sizes in
   test_oracle_roundtrip.py): `bin_offset` is the exclusive cumsum of the per-bin counts of the generator's clusters, the
   attached part of every bin is the generator's clusters in a stable sort by bin, the unattached
   part is the generator's unattached clusters of the bin sorted by the encoder's tuple (C6).  No expected value comes from
   the CUDA path.
2. SAMPLED tracks (random ones, the longest ones, the first and the last) go through the ORACLE one by one: the oracle's
   encoder, fed with the generator's clusters of the track, must produce the bytes the GPU encoder left in the workload
   (so the oracle's input is its own), and the oracle's decode of them must equal the records the GPU wrote at the
   canonical positions of the track's clusters.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu
BZ = 0.5


def _decode_like_bench(geo, arrays):
    import torch
    from paper_2411_02206_b200 import tmd as T
    device = arrays["trk_ncl"].device
    n_trk, n_att, n_un = (int(arrays[k].shape[0]) for k in ("trk_ncl", "a_qtot", "u_qtot"))
    ctx = T.tmd_create(geo, BZ)
    try:
        clusters = torch.full(((n_att + n_un) * 4,), -0x11111112, dtype=torch.int32, device=device)
        bin_offset = torch.empty(geo.n_bins + 1, dtype=torch.int32, device=device)
        ws = torch.empty(T.tmd_workspace_bytes(ctx, n_trk, n_att, n_un), dtype=torch.uint8, device=device)
        T.tmd_decode(ctx, T.make_compressed(arrays), T.make_output(clusters, bin_offset, ws), 0, torch.cuda.current_stream().cuda_stream)
        torch.cuda.synchronize()
    finally:
        T.tmd_destroy(ctx)
    return clusters.view(-1, 4), bin_offset


@pytest.mark.parametrize("name", ["c2", "c3", "c4"])
def test_full_time_frame(name):
    import torch
    import bench
    from oracle import tmd_oracle as O
    from tmd_inputs import physical as ph, timeframe as tf
    from tmd_inputs.layout import CLUSTER_DTYPE

    dev = torch.device("cuda", 0)
    geo, arrays, truth = bench.build_workload(name, dev, keep_truth=True)
    n_trk, n_att, n_un, n_bins = truth.n_tracks, truth.n_attached, int(arrays["u_qtot"].shape[0]), geo.n_bins
    got, got_bo = _decode_like_bench(geo, arrays)

    # ---- 1. every record, from the definition (torch library routines on the generator's clusters)
    w3 = truth.att[:, 3]
    bins = (((w3 >> 16) & 0xFF) * geo.n_rows + ((w3 >> 8) & 0xFF)).to(torch.int32)
    att_cnt = torch.bincount(bins, minlength=n_bins)
    u_cnt = arrays["u_bin_count"].to(torch.int64)
    want_bo = torch.zeros(n_bins + 1, dtype=torch.int64, device=dev)
    want_bo[1:] = torch.cumsum(att_cnt + u_cnt, 0)
    assert torch.equal(got_bo.to(torch.int64) & 0xFFFFFFFF, want_bo), "bin_offset"
    order = torch.sort(bins, stable=True).indices                     # canonical order of the attached clusters (C5)
    u_start = torch.cumsum(u_cnt, 0) - u_cnt
    dest = torch.empty(n_att, dtype=torch.int64, device=dev)           # canonical position of attached cluster g
    dest[order] = torch.arange(n_att, device=dev) + u_start[bins[order].long()]
    del order
    bad = (got[dest] != truth.att).any(dim=1)
    assert not bool(bad.any()), f"{int(bad.sum())} attached records differ; first g = {int(bad.nonzero()[0])}"
    del bad
    # unattached: the generator's clusters in the encoder's order -- per bin ascending by (time, pad, qtot, qmax, sigpad,
    # sigtime, flags) (C6), two stable library sorts -- appended after the bin's attached clusters (C5)
    un = truth.un.to(torch.int64)
    u0, u1, u2, u3 = (un[:, k] & 0xFFFFFFFF for k in range(4))
    ubin_any = ((u3 >> 16) & 0xFF) * geo.n_rows + ((u3 >> 8) & 0xFF)
    assert torch.equal(torch.bincount(ubin_any, minlength=n_bins), u_cnt), "u_bin_count"
    key_lo = ((u1 >> 16) << 40) | ((u2 & 0xFFFF) << 24) | (((u2 >> 16) & 0xFF) << 16) | (((u2 >> 24) & 0xFF) << 8) | (u3 & 0xFF)
    key_hi = (ubin_any << 48) | (u0 << 16) | (u1 & 0xFFFF)
    o1 = torch.sort(key_lo, stable=True).indices
    o2 = torch.sort(key_hi[o1], stable=True).indices
    order_u = o1[o2]
    del un, u0, u1, u2, u3, key_lo, key_hi, o1, o2
    want_u = truth.un[order_u]
    ubin = ubin_any[order_u]
    del order_u, ubin_any
    i_in = torch.arange(n_un, device=dev) - u_start[ubin]
    udest = want_bo[ubin] + att_cnt[ubin] + i_in
    bad = (got[udest] != want_u).any(dim=1)
    assert not bool(bad.any()), f"{int(bad.sum())} unattached records differ"
    del bad, want_u, udest, ubin, i_in

    # ---- 2. sampled tracks through the oracle, one by one
    rng = np.random.default_rng(7)
    ncl = (truth.trk_ncl.to(torch.int64) & 0xFFFF)
    off = torch.cumsum(ncl, 0) - ncl
    longest = torch.topk(ncl, 16).indices.cpu().numpy()
    sample = np.unique(np.concatenate((rng.integers(0, n_trk, 400), longest, [0, n_trk - 1])))
    h_off, h_ncl = off.cpu().numpy(), ncl.cpu().numpy()
    res_fields = ("a_rowdiff", "a_secleg", "a_padres", "a_timeres")
    for t in sample:
        g0, n = int(h_off[t]), int(h_ncl[t])
        att = truth.att[g0:g0 + n].cpu().numpy().view(CLUSTER_DTYPE).reshape(-1)
        leg = truth.leg[g0:g0 + n].cpu().numpy()
        comp = O.encode(geo, BZ, np.array([n], np.uint16), truth.trk_qptf[t:t + 1].cpu().numpy(), att, leg, np.zeros(0, CLUSTER_DTYPE))
        r0 = g0 - int(t)
        for k in res_fields:                                            # the GPU-encoded streams are the oracle's own bytes
            mine = arrays[k][r0:r0 + n - 1].cpu().numpy().view(getattr(comp, k).dtype)
            assert np.array_equal(mine, getattr(comp, k)), f"track {t}: {k}"
        for k in ("trk_qpt", "trk_row0", "trk_sec0", "trk_pad0", "trk_time0"):
            assert arrays[k][t:t + 1].cpu().numpy().view(getattr(comp, k).dtype)[0] == getattr(comp, k)[0], f"track {t}: {k}"
        d = O.decode_track(geo, BZ, int(comp.trk_qpt[0]), int(comp.trk_sec0[0]), int(comp.trk_row0[0]), int(comp.trk_pad0[0]),
                           int(comp.trk_time0[0]), comp.a_rowdiff, comp.a_secleg, comp.a_padres, comp.a_timeres)
        rec = got[dest[g0:g0 + n]].cpu().numpy().view(CLUSTER_DTYPE).reshape(-1)
        for f, key in (("sector", "sec"), ("row", "row"), ("pad", "P"), ("time", "T")):
            assert np.array_equal(rec[f], d[key]), f"track {t}: {f}"
        for f in ("qtot", "qmax", "sigpad", "sigtime", "flags"):
            assert np.array_equal(rec[f], att[f]), f"track {t}: {f}"


# ------------------------------------------------------------------------------------------------ the full oracle at full size
def _host_gb_available() -> float:
    import psutil
    return psutil.virtual_memory().available / 2 ** 30


def _upload(comp):
    from gpu_util import _as_torch
    from tmd_inputs.layout import COMPRESSED_FIELDS
    return {k: _as_torch(np.ascontiguousarray(getattr(comp, k))).cuda() for k in COMPRESSED_FIELDS}


def _compare_with_oracle(geo, comp, tag):
    """tmd_decode in the launch configuration bench.py times (flags 0, no probes) against orc_decode: every record."""
    from oracle import tmd_oracle as O
    from tmd_inputs.layout import CLUSTER_DTYPE
    got, got_bo = _decode_like_bench(geo, _upload(comp))
    want, want_bo, _ = O.decode(geo, BZ, comp)
    assert np.array_equal(got_bo.cpu().numpy().view(np.uint32), want_bo), f"{tag}: bin_offset"
    got = got.cpu().numpy().view(CLUSTER_DTYPE).reshape(-1)
    if got.tobytes() != want.tobytes():
        for f in want.dtype.names:
            bad = np.nonzero(got[f] != want[f])[0]
            assert bad.size == 0, f"{tag}: {bad.size} records differ in {f}; first at {int(bad[0])}: got {got[f][bad[0]]} want {want[f][bad[0]]}"
        raise AssertionError(f"{tag}: bytes differ")


# host memory the oracle side needs (truth + compressed SoA + two outputs), GB
@pytest.mark.parametrize("name,need_gb", [("c2", 8), ("c3", 30), ("c4", 14)])
def test_full_time_frame_against_the_full_oracle(name, need_gb):
    """BASELINE.json north_star: "bit-exact agreement with the CPU oracle on all five configs".  The whole frame (attached
    AND unattached clusters) goes through the ORACLE ENCODER (configs: "encoded by the oracle encoder"), tmd_decode runs as
    bench.py runs it, and every output record and bin offset is compared with orc_decode.  The GPU encoder is compared
    with the oracle's bytes on the way (it is what builds bench.py's timed workload)."""
    import torch
    from oracle import tmd_oracle as O
    from paper_2411_02206_b200 import tmd as T
    from tmd_inputs import build_geometry, timeframe as tf
    from tmd_inputs.layout import CLUSTER_DTYPE

    if _host_gb_available() < need_gb:
        pytest.skip(f"needs {need_gb} GB of host memory for the oracle side, {_host_gb_available():.0f} GB available")
    dev = torch.device("cuda", 0)
    geo = build_geometry(36)
    mk, n_un, single = tf.WORKLOADS[name]
    cfg = mk()
    truth = tf.generate_truth(cfg, geo, dev, batch=2_000_000)
    un = tf.generate_unattached_truth(geo, n_un, cfg.seed, dev, "inv_x", single)
    comp = O.encode(geo, BZ, truth.trk_ncl.cpu().numpy().view(np.uint16), truth.trk_qptf.cpu().numpy(),
                    truth.att.cpu().numpy().view(CLUSTER_DTYPE).reshape(-1), truth.leg.cpu().numpy(),
                    un.cpu().numpy().view(CLUSTER_DTYPE).reshape(-1))
    del un
    # the library's encoder on the same truth: the oracle encoder's bytes
    ctx = T.tmd_create(geo, BZ)
    try:
        tdt = {"<u2": torch.int16, "i1": torch.int8, "u1": torch.uint8, "<u4": torch.int32}
        mine = {k: torch.zeros(len(getattr(comp, k)), dtype=tdt[dt], device=dev) for k, dt in T.COMPRESSED_ARRAYS
                if k.startswith(("trk_", "a_")) and k != "trk_ncl"}
        ws = torch.empty(T.tmd_workspace_bytes(ctx, truth.n_tracks, truth.n_attached, 0), dtype=torch.uint8, device=dev)
        T.tmd_encode_attached(ctx, truth.trk_ncl, truth.trk_qptf, truth.att, truth.leg, mine, ws, torch.cuda.current_stream().cuda_stream)
        for k, v in mine.items():
            assert np.array_equal(v.cpu().numpy().view(getattr(comp, k).dtype), getattr(comp, k)), f"{name}: GPU encoder, {k}"
        del mine, ws
    finally:
        T.tmd_destroy(ctx)
    del truth
    torch.cuda.empty_cache()
    _compare_with_oracle(geo, comp, name)


def test_random_bytes_at_the_full_frame_chunk_size():
    """>= 97 M attached clusters of random bytes: the library picks chunk_shift = 15 (32768-record chunks, multi-trip loops in
    the scatter, the multi-run path of the rank kernel on every group) -- the launch configuration of c2..c4, which the small
    adversarial inputs never reach.  Against the full oracle."""
    from tmd_inputs import build_geometry
    from tmd_inputs.adversarial import random_compressed
    if _host_gb_available() < 12:
        pytest.skip("needs 12 GB of host memory")
    geo = build_geometry(36)
    c = random_compressed(geo, 1_000_000, 3_000_000, seed=61, max_ncl=199)
    assert c.n_attached >= 97_000_000
    _compare_with_oracle(geo, c, "random bytes, shift 15")


@pytest.mark.parametrize("n_tracks", [120_000, 220_000, 400_000])
def test_random_bytes_at_the_intermediate_chunk_sizes(n_tracks):
    """~12 M, ~22 M and ~40 M attached clusters of random bytes: on a 148-SM device the library's chunk-size rule
    (csrc/tmd_api.cu, layout) picks chunks of 2^12, 2^13 and 2^14 records for them -- the sizes between the small adversarial inputs
    (2^11) and the full frames (2^15).  Against the full oracle."""
    from tmd_inputs import build_geometry
    from tmd_inputs.adversarial import random_compressed
    geo = build_geometry(36)
    c = random_compressed(geo, n_tracks, n_tracks // 2, seed=70 + n_tracks // 100_000, max_ncl=199)
    _compare_with_oracle(geo, c, f"random bytes, {c.n_attached} attached")


def test_whole_chunks_in_one_bin_at_the_full_frame_chunk_size():
    """Tracks of 65 535 clusters that never leave their first bin, half of them sharing one bin: whole 32768-record chunks
    fall into a single bin (u16 histogram / rank / start entries at their limit).  Against the full oracle."""
    from tmd_inputs import build_geometry
    from tmd_inputs.adversarial import degenerate_same_bin
    if _host_gb_available() < 12:
        pytest.skip("needs 12 GB of host memory")
    geo = build_geometry(36)
    ncl = np.full(1500, 65535, np.uint16)
    ncl[::97] = 1
    ncl[5::211] = 32769
    extra = int(97_500_000 - ncl.astype(np.int64).sum())
    if extra > 0:
        ncl = np.concatenate((ncl, np.full(extra // 65535 + 1, 65535, np.uint16)))
    c = degenerate_same_bin(geo, ncl, 62, n_un=10_000)
    assert c.n_attached >= 97_000_000
    _compare_with_oracle(geo, c, "one bin, shift 15")


def test_full_c2_container_in_clusters_out():
    """The whole chain at time-frame size: oracle encoder -> ORACLE rANS coder -> container in pinned host memory ->
    tmd_decode_container_host_async (upload, GPU entropy decode, track-model decode, download) -> every record and bin offset
    against orc_decode.  No input of the library comes from the library."""
    import torch
    from oracle import tmd_ans as ANS, tmd_oracle as O
    from paper_2411_02206_b200 import tmd as T
    from tmd_inputs import build_geometry, timeframe as tf
    from tmd_inputs.layout import CLUSTER_DTYPE

    if _host_gb_available() < 12:
        pytest.skip(f"needs 12 GB of host memory for the oracle side, {_host_gb_available():.0f} GB available")
    dev = torch.device("cuda", 0)
    geo = build_geometry(36)
    mk, n_un, single = tf.WORKLOADS["c2"]
    cfg = mk()
    truth = tf.generate_truth(cfg, geo, dev, batch=2_000_000)
    un = tf.generate_unattached_truth(geo, n_un, cfg.seed, dev, "inv_x", single)
    comp = O.encode(geo, BZ, truth.trk_ncl.cpu().numpy().view(np.uint16), truth.trk_qptf.cpu().numpy(),
                    truth.att.cpu().numpy().view(CLUSTER_DTYPE).reshape(-1), truth.leg.cpu().numpy(),
                    un.cpu().numpy().view(CLUSTER_DTYPE).reshape(-1))
    del truth, un
    torch.cuda.empty_cache()
    blob = torch.from_numpy(ANS.encode_container(comp)).pin_memory()
    assert blob.numel() < comp.nbytes() / 1.5                      # it is a compressed container
    want_cl, want_bo, _ = O.decode(geo, BZ, comp)
    n = comp.n_attached + comp.n_unattached
    hc = torch.full((n * 16,), 0xEE, dtype=torch.uint8).pin_memory()
    hb = torch.zeros(geo.n_bins + 1, dtype=torch.int32).pin_memory()
    ctx = T.tmd_create(geo, BZ)
    try:
        T.tmd_decode_container_host_async(ctx, blob, T.make_output(hc, hb), 0, 0)
        T.tmd_host_wait(ctx, 0)
    finally:
        T.tmd_destroy(ctx)
    assert np.array_equal(hb.numpy().view(np.uint32), want_bo)
    got = hc.numpy().view(CLUSTER_DTYPE)
    if got.tobytes() != want_cl.tobytes():
        for f in want_cl.dtype.names:
            d = np.nonzero(got[f] != want_cl[f])[0]
            assert d.size == 0, f"{d.size} records differ in {f}; first at {int(d[0])}"
        raise AssertionError("bytes differ")
