"""`-m gpu` parity: the CUDA library (through its C ABI) against the CPU oracle, element by element.

Bar (BASELINE.json north_star): bit-exact on every integer cluster field in canonical order, bin offsets equal, and the
fp32 track-state probes equal to the oracle's at 0 ULP (no FMA contraction on either side).  Inputs are seeded and
synthetic: helix events encoded by the oracle encoder (configs c0, c1 full size, c2/c4-shaped), adversarial random bytes
and degenerate cases.
"""
import numpy as np
import pytest

from oracle import tmd_oracle as O
from tmd_inputs import build_geometry, physical as ph
from tmd_inputs.adversarial import degenerate_same_bin, random_compressed
from tmd_inputs.layout import Compressed

from gpu_util import first_mismatch, gpu_decode

pytestmark = pytest.mark.gpu
BZ = 0.5

PHYS = {
    "c0": (lambda: ph.config0(), 2),
    "c1": (lambda: ph.config1(), 36),
    "c2_like": (lambda: ph.config2_like(6000, 90_000), 36),
    "c4_like": (lambda: ph.config4_like(40_000, 100_000), 36),
}


def assert_same(got, want):
    g_cl, g_bo, g_pr = got
    w_cl, w_bo, w_pr = want
    assert np.array_equal(g_bo, w_bo), "bin_offset: " + first_mismatch(g_bo, w_bo)
    for f in w_cl.dtype.names:
        assert np.array_equal(g_cl[f], w_cl[f]), f"{f}: " + first_mismatch(g_cl[f], w_cl[f])
    assert g_cl.tobytes() == w_cl.tobytes()
    if w_pr is not None:
        nan = np.isnan(w_pr.view(np.float32))            # NaN payloads are not compared (reading 15)
        assert np.array_equal(np.isnan(g_pr.view(np.float32)), nan)
        ulp = np.abs(g_pr.astype(np.int64) - w_pr.astype(np.int64))[~nan]
        assert ulp.max(initial=0) == 0, f"probe state deviates by up to {ulp.max()} ULP in {np.count_nonzero(ulp)} values"


@pytest.fixture(scope="module", params=list(PHYS))
def phys_case(request):
    mk, nsec = PHYS[request.param]
    geo = build_geometry(nsec)
    ev = ph.generate_event(mk(), geo)
    comp = O.encode(geo, BZ, ev.trk_ncl, ev.trk_qptf, ev.att, ev.leg, ev.un)
    return request.param, geo, ev, comp


def test_physical_events_match_oracle(phys_case):
    name, geo, ev, comp = phys_case
    assert_same(gpu_decode(geo, BZ, comp, probe_step=0xFFFFFFFF), O.decode(geo, BZ, comp, probe_step=0xFFFFFFFF))


def test_physical_events_round_trip(phys_case):
    # decode(encode(x)) == canonical(x): the GPU decoder restores the generator's clusters
    name, geo, ev, comp = phys_case
    cl, bo, _ = gpu_decode(geo, BZ, comp)
    want, want_bo = ph.canonical(ev, geo)
    assert np.array_equal(bo, want_bo) and cl.tobytes() == want.tobytes()


@pytest.mark.parametrize("step", [0, 1, 7, "half"])
def test_probes_at_intermediate_steps(phys_case, step):
    name, geo, ev, comp = phys_case
    if name not in ("c0", "c4_like"):
        pytest.skip("probe sweep on two cases")
    s = int(np.median(comp.trk_ncl)) // 2 if step == "half" else step
    assert_same(gpu_decode(geo, BZ, comp, probe_step=s), O.decode(geo, BZ, comp, probe_step=s))


def test_host_entry_point_matches(phys_case):
    name, geo, ev, comp = phys_case
    if name != "c0":
        pytest.skip("one case")
    assert_same(gpu_decode(geo, BZ, comp, probe_step=3, via_host=True), O.decode(geo, BZ, comp, probe_step=3))


@pytest.mark.parametrize("seed,n_tracks,n_un,max_ncl", [(1, 300, 4000, 40), (2, 1, 0, 40), (3, 50, 0, 40), (4, 0, 100, 40),
                                                       (5, 20_000, 150_000, 200), (6, 3000, 0, 1000)])
def test_adversarial_random_bytes(seed, n_tracks, n_un, max_ncl):
    geo = build_geometry(36)
    c = random_compressed(geo, n_tracks, n_un, seed, max_ncl=max_ncl)
    assert_same(gpu_decode(geo, BZ, c, probe_step=0xFFFFFFFF), O.decode(geo, BZ, c, probe_step=0xFFFFFFFF))


@pytest.mark.parametrize("tail", [0, 1, 5, 15, 16, 17, 33, 70])
def test_every_track_length_at_every_staging_phase(tail):
    """The decode kernel stages a track's residuals in 16-byte cells of per-stream rings: which cells are
    staged before the loop, which are requested inside it and which are never needed depends on the track's length and on
    its first residual index modulo 16.  Lengths 1..100 in a shuffled order put every length at many phases; `tail` is the
    length of the LAST track, so that the arrays end in the middle of a cell for several remainders (the zero-filled copy
    that must not read past the arrays) with the last track inside or beyond its pre-staged cells."""
    geo = build_geometry(36)
    rng = np.random.default_rng(100 + tail)
    ncl = np.concatenate([rng.permutation(np.arange(1, 101)) for _ in range(24)] + [np.array([tail + 1])]).astype(np.uint16)
    c = random_compressed(geo, 0, 300, 200 + tail, ncl=ncl)
    assert_same(gpu_decode(geo, BZ, c, probe_step=0xFFFFFFFF), O.decode(geo, BZ, c, probe_step=0xFFFFFFFF))


def test_empty_and_one_sided_inputs():
    geo = build_geometry(36)
    c = Compressed.empty(0, 0, 0, geo.n_bins)
    cl, bo, _ = gpu_decode(geo, BZ, c)
    assert len(cl) == 0 and np.all(bo == 0)
    c = random_compressed(geo, 0, 0, 11, ncl=np.ones(500, np.uint16))       # only single-cluster tracks: no residuals at all
    assert_same(gpu_decode(geo, BZ, c), O.decode(geo, BZ, c))


def test_tracks_longer_than_a_chunk_window():
    # trk_ncl up to the format's maximum (65535): tracks straddle several 32768-cluster windows of the rank pass
    geo = build_geometry(36)
    ncl = np.array([5, 65535, 1, 40000, 32768, 32767, 3, 152, 65535, 9], np.uint16)
    c = random_compressed(geo, 0, 1000, 12, ncl=ncl)
    assert_same(gpu_decode(geo, BZ, c, probe_step=0xFFFFFFFF), O.decode(geo, BZ, c, probe_step=0xFFFFFFFF))


def test_degenerate_all_clusters_in_one_bin():
    geo = build_geometry(36)
    rng = np.random.default_rng(3)
    ncl = np.concatenate((rng.integers(1, 300, 400), [20000, 1, 1, 9000])).astype(np.uint16)
    c = degenerate_same_bin(geo, ncl, 13, n_un=500)
    assert_same(gpu_decode(geo, BZ, c), O.decode(geo, BZ, c))


def test_unattached_skewed_bins():
    geo = build_geometry(36)
    rng = np.random.default_rng(21)
    counts = rng.poisson(2.0, geo.n_bins).astype(np.uint32)
    counts[17] = 300_000           # one bin much larger than a tile
    counts[18] = 1
    counts[geo.n_bins - 1] = 5000
    n = int(counts.sum())
    c = random_compressed(geo, 10, 0, 22)
    u = Compressed.empty(c.n_tracks, c.n_attached, n, geo.n_bins)
    for k in ("trk_ncl", "trk_qpt", "trk_row0", "trk_sec0", "trk_pad0", "trk_time0", "a_qtot", "a_qmax", "a_flags", "a_sigpad",
              "a_sigtime", "a_rowdiff", "a_secleg", "a_padres", "a_timeres"):
        getattr(u, k)[:] = getattr(c, k)
    u.u_bin_count[:] = counts
    u.u_paddiff[:] = rng.integers(0, 65536, n); u.u_timediff[:] = rng.integers(0, 2 ** 32, n)
    u.u_qtot[:] = rng.integers(0, 65536, n); u.u_qmax[:] = rng.integers(0, 65536, n)
    u.u_flags[:] = rng.integers(0, 256, n); u.u_sigpad[:] = rng.integers(0, 256, n); u.u_sigtime[:] = rng.integers(0, 256, n)
    assert_same(gpu_decode(geo, BZ, u), O.decode(geo, BZ, u))


def test_validate_flag_reports_corrupt_counts():
    from paper_2411_02206_b200 import tmd as T
    geo = build_geometry(36)
    c = random_compressed(geo, 100, 100, 31)
    assert_same(gpu_decode(geo, BZ, c, flags=T.TMD_VALIDATE), O.decode(geo, BZ, c))
    bad = random_compressed(geo, 100, 100, 31)
    bad.u_bin_count[5] += 1
    bad.u_bin_count[6] = max(int(bad.u_bin_count[6]), 1) - 1 if bad.u_bin_count[6] > 0 else 0
    if int(bad.u_bin_count.sum()) != bad.n_unattached:
        with pytest.raises(T.TmdError) as e:
            gpu_decode(geo, BZ, bad, flags=T.TMD_VALIDATE)
        assert e.value.status == T.TMD_ERR_CORRUPT
    bad = random_compressed(geo, 100, 100, 31)
    bad.trk_row0[7] = 200
    with pytest.raises(T.TmdError) as e:
        gpu_decode(geo, BZ, bad, flags=T.TMD_VALIDATE)
    assert e.value.status == T.TMD_ERR_CORRUPT
    # config 0 geometry (2 output sectors): a decoded sector >= 2 is reported (reading 20)
    geo2 = build_geometry(2)
    c2 = random_compressed(geo2, 50, 10, 32, n_sectors_in=36)
    with pytest.raises(T.TmdError) as e:
        gpu_decode(geo2, BZ, c2, flags=T.TMD_VALIDATE)
    assert e.value.status == T.TMD_ERR_CORRUPT


def test_gpu_encoder_matches_oracle_encoder(phys_case):
    # tmd_encode_attached (the synchronous-side step) produces the oracle encoder's bytes
    import torch
    from paper_2411_02206_b200 import tmd as T
    from gpu_util import _as_torch
    name, geo, ev, comp = phys_case
    ctx = T.tmd_create(geo, BZ)
    try:
        dev = lambda a: _as_torch(np.ascontiguousarray(a)).cuda()
        att = torch.from_numpy(np.ascontiguousarray(ev.att).view(np.int32).reshape(-1, 4)).cuda()
        out = {}
        for k in ("trk_qpt", "trk_row0", "trk_sec0", "trk_pad0", "trk_time0", "a_qtot", "a_qmax", "a_flags", "a_sigpad", "a_sigtime",
                  "a_rowdiff", "a_secleg", "a_padres", "a_timeres"):
            out[k] = torch.zeros_like(dev(getattr(comp, k)))
        ws = torch.empty(T.tmd_workspace_bytes(ctx, comp.n_tracks, comp.n_attached, 0), dtype=torch.uint8, device="cuda")
        T.tmd_encode_attached(ctx, dev(ev.trk_ncl), dev(ev.trk_qptf), att, dev(ev.leg), out, ws, torch.cuda.current_stream().cuda_stream)
        for k, v in out.items():
            want = getattr(comp, k)
            got = v.cpu().numpy().view(want.dtype)
            assert np.array_equal(got, want), f"{k}: " + first_mismatch(got, want)
    finally:
        T.tmd_destroy(ctx)


def test_bench_workload_builder_matches_oracle():
    # the path bench.py times: torch cluster truth -> GPU encoder (attached + unattached) -> GPU decoder.  The oracle gets the
    # generator's clusters and its OWN encoder's bytes; the GPU encoder's bytes must be the same, then both decoders must agree.
    import torch
    import bench
    from tmd_inputs.layout import CLUSTER_DTYPE, COMPRESSED_FIELDS
    geo, arrays, truth = bench.build_workload("c1", torch.device("cuda", 0), keep_truth=True)
    att = truth.att.cpu().numpy().view(CLUSTER_DTYPE).reshape(-1)
    comp = O.encode(geo, BZ, truth.trk_ncl.cpu().numpy().view(np.uint16), truth.trk_qptf.cpu().numpy(), att, truth.leg.cpu().numpy(),
                    truth.un.cpu().numpy().view(CLUSTER_DTYPE).reshape(-1))
    assert comp.n_tracks == 10_000 and 1.1e6 < comp.n_attached < 1.4e6 and 2.9e5 < comp.n_unattached < 3.1e5
    for k, (dt, which) in COMPRESSED_FIELDS.items():
        mine = arrays[k].cpu().numpy().view(np.dtype(dt))
        assert np.array_equal(mine, getattr(comp, k)), f"GPU encoder, {k}: " + first_mismatch(mine, getattr(comp, k))
    assert_same(gpu_decode(geo, BZ, comp, probe_step=0xFFFFFFFF), O.decode(geo, BZ, comp, probe_step=0xFFFFFFFF))


def test_pipelined_host_entry_points_match():
    # tmd_decode_host_async / tmd_host_wait: frames alternate between the two slots; each result equals the oracle's
    import torch
    from paper_2411_02206_b200 import tmd as T
    from tmd_inputs.layout import CLUSTER_DTYPE, COMPRESSED_FIELDS
    from gpu_util import _as_torch
    geo = build_geometry(36)
    frames = [random_compressed(geo, 3000, 20_000, 41, max_ncl=200), random_compressed(geo, 500, 90_000, 42, max_ncl=60),
              random_compressed(geo, 4000, 1000, 43, max_ncl=150)]
    want = [O.decode(geo, BZ, c) for c in frames]
    ctx = T.tmd_create(geo, BZ)
    try:
        held = []
        for i, c in enumerate(frames):
            h_in = {k: _as_torch(np.ascontiguousarray(getattr(c, k))).pin_memory() for k in COMPRESSED_FIELDS}
            n = c.n_attached + c.n_unattached
            hc = torch.zeros(n * 16, dtype=torch.uint8).pin_memory()
            hb = torch.zeros(geo.n_bins + 1, dtype=torch.int32).pin_memory()
            held.append((h_in, hc, hb))
            T.tmd_decode_host_async(ctx, T.make_compressed(h_in), T.make_output(hc, hb), 0, i % T.TMD_HOST_SLOTS)
        for s_ in range(T.TMD_HOST_SLOTS):
            T.tmd_host_wait(ctx, s_)
        for (h_in, hc, hb), (w_cl, w_bo, _) in zip(held, want):
            assert np.array_equal(hb.numpy().view(np.uint32), w_bo)
            assert hc.numpy().view(CLUSTER_DTYPE).tobytes() == w_cl.tobytes()
        with pytest.raises(T.TmdError):
            T.tmd_decode_host_async(ctx, T.make_compressed(held[0][0]), T.make_output(held[0][1], held[0][2]), T.TMD_VALIDATE, 0)
    finally:
        T.tmd_destroy(ctx)


def test_timing_and_validate_flags_do_not_change_the_result():
    # TMD_TIMING (event pairs around the kernels) is the mode bench.py's per-kernel pass uses
    import torch
    from paper_2411_02206_b200 import tmd as T
    geo = build_geometry(36)
    c = random_compressed(geo, 5000, 60_000, 51, max_ncl=180)
    want = O.decode(geo, BZ, c)
    for flags in (T.TMD_TIMING, T.TMD_VALIDATE, T.TMD_TIMING | T.TMD_VALIDATE):
        assert_same(gpu_decode(geo, BZ, c, flags=flags), want)
    ctx = T.tmd_create(geo, BZ)
    try:
        from gpu_util import _as_torch
        from tmd_inputs.layout import COMPRESSED_FIELDS
        dev = {k: _as_torch(np.ascontiguousarray(getattr(c, k))).cuda() for k in COMPRESSED_FIELDS}
        n = c.n_attached + c.n_unattached
        out = T.make_output(torch.empty(n * 16, dtype=torch.uint8, device="cuda"), torch.empty(geo.n_bins + 1, dtype=torch.int32, device="cuda"),
                            torch.empty(T.tmd_workspace_bytes(ctx, c.n_tracks, c.n_attached, c.n_unattached), dtype=torch.uint8, device="cuda"))
        T.tmd_decode(ctx, T.make_compressed(dev), out, T.TMD_TIMING, torch.cuda.current_stream().cuda_stream)
        times = dict(T.tmd_kernel_times(ctx))
        assert T.tmd_last_launch_count(ctx) == len(times) == 12
        assert {"track_decode", "rank", "scatter", "unattached", "bin_offsets"} <= set(times) and all(v >= 0 for v in times.values())
    finally:
        T.tmd_destroy(ctx)


def test_batch_of_frames_equals_frame_by_frame():
    # tmd_decode_batch: frames of very different sizes -- physical events, random bytes, a frame without
    # tracks, one without unattached clusters, an empty one -- decoded by ONE launch sequence; every frame against the oracle
    import torch
    from paper_2411_02206_b200 import tmd as T
    from gpu_util import _as_torch
    from tmd_inputs.layout import CLUSTER_DTYPE, COMPRESSED_FIELDS
    geo = build_geometry(36)
    ev = ph.generate_event(ph.config2_like(1500, 20_000, seed=71), geo)
    frames = [O.encode(geo, BZ, ev.trk_ncl, ev.trk_qptf, ev.att, ev.leg, ev.un),
              random_compressed(geo, 3000, 20_000, 72, max_ncl=200), random_compressed(geo, 0, 5000, 73),
              random_compressed(geo, 700, 0, 74, max_ncl=90), Compressed.empty(0, 0, 0, geo.n_bins),
              random_compressed(geo, 0, 0, 75, ncl=np.array([65535, 1, 40000, 7], np.uint16)),
              degenerate_same_bin(geo, np.full(300, 500, np.uint16), 76, n_un=100)]
    frames += [random_compressed(geo, 50 + 37 * i, 400 * i, 80 + i, max_ncl=30 + 10 * i) for i in range(12)]   # > one table chunk
    want = [O.decode(geo, BZ, c, probe_step=2) for c in frames]
    ctx = T.tmd_create(geo, BZ)
    try:
        comps, outs, held = [], [], []
        for i, c in enumerate(frames):
            dev = {k: _as_torch(np.ascontiguousarray(getattr(c, k))).cuda() for k in COMPRESSED_FIELDS}
            n = c.n_attached + c.n_unattached
            d_cl = torch.full((max(n, 1) * 16,), 0xEE, dtype=torch.uint8, device="cuda")
            d_bo = torch.zeros(geo.n_bins + 1, dtype=torch.int32, device="cuda")
            d_pr = torch.zeros(max(c.n_tracks, 1) * 6, dtype=torch.int32, device="cuda") if i % 2 == 0 else None   # probes on some frames only
            ws = torch.empty(T.tmd_workspace_bytes(ctx, c.n_tracks, c.n_attached, c.n_unattached), dtype=torch.uint8, device="cuda")
            held.append((dev, d_cl, d_bo, d_pr, ws))
            comps.append(T.make_compressed(dev)); outs.append(T.make_output(d_cl, d_bo, ws, d_pr, 2))
        T.tmd_decode_batch(ctx, T.make_batch(comps, outs), 0, torch.cuda.current_stream().cuda_stream)
        torch.cuda.synchronize()
        for i, (c, (dev, d_cl, d_bo, d_pr, ws), (w_cl, w_bo, w_pr)) in enumerate(zip(frames, held, want)):
            n = c.n_attached + c.n_unattached
            got = (d_cl.cpu().numpy()[: n * 16].view(CLUSTER_DTYPE).copy(), d_bo.cpu().numpy().view(np.uint32).copy(),
                   d_pr.cpu().numpy().view(np.uint32)[: c.n_tracks * 6].reshape(-1, 6).copy() if d_pr is not None else None)
            assert_same(got, (w_cl, w_bo, w_pr if d_pr is not None else None))
        with pytest.raises(T.TmdError):                      # TMD_VALIDATE synchronises: not accepted for a batch
            T.tmd_decode_batch(ctx, T.make_batch(comps, outs), T.TMD_VALIDATE, 0)
        # TMD_TIMING on a batch whose frame table needs many upload launches (19 frames x 11 = 209 frames -> 27 launches, more
        # than the TMD_MAX_KERNELS event pairs): the upload is one row and every decode kernel is still reported
        more = []
        for rep in range(10):                                # the same inputs again, every frame with outputs and workspace of its own
            for c, (dev, d_cl, d_bo, d_pr, ws) in zip(frames, held):
                bufs = (torch.empty_like(d_cl), torch.empty_like(d_bo), torch.empty_like(ws))
                held.append(bufs)                            # tmd_output holds addresses only: keep the tensors alive
                more.append(T.make_output(*bufs))
        many = T.make_batch(comps * 11, outs + more)
        T.tmd_decode_batch(ctx, many, T.TMD_TIMING, torch.cuda.current_stream().cuda_stream)
        rows = T.tmd_kernel_times(ctx)
        names = [r[0] for r in rows]
        assert names.count("store_frames") == 1 and names[0] == "store_frames" and names[-1] == "scatter" and len(rows) == 13
        assert T.tmd_last_launch_count(ctx) == 12 + 27
        torch.cuda.synchronize()
    finally:
        T.tmd_destroy(ctx)


def test_validate_sums_track_lengths_in_64_bits():
    # 70000 tracks of 65535 clusters sum to 4 587 450 000 = 292 482 704 mod 2^32: an input that declares n_attached =
    # 292 482 704 must be rejected (a 32-bit sum wraps onto the declared value and the decode would run off the workspace)
    import torch
    from paper_2411_02206_b200 import tmd as T
    geo = build_geometry(36)
    n_trk, n_att = 70_000, 292_482_704
    assert (n_trk * 65535) % 2 ** 32 == n_att
    from tmd_inputs.layout import COMPRESSED_FIELDS
    lens = {"n_tracks": n_trk, "n_attached": n_att, "n_residuals": n_att - n_trk, "n_unattached": 0, "n_bins": geo.n_bins}
    tdt = {"<u2": torch.int16, "i1": torch.int8, "u1": torch.uint8, "<u4": torch.int32}
    dev = {k: torch.zeros(lens[which], dtype=tdt[dt], device="cuda") for k, (dt, which) in COMPRESSED_FIELDS.items()}
    dev["trk_ncl"].fill_(-1)                                 # 0xFFFF = 65535
    ctx = T.tmd_create(geo, BZ)
    try:
        out = T.make_output(torch.empty(n_att * 16, dtype=torch.uint8, device="cuda"), torch.empty(geo.n_bins + 1, dtype=torch.int32, device="cuda"),
                            torch.empty(T.tmd_workspace_bytes(ctx, n_trk, n_att, 0), dtype=torch.uint8, device="cuda"))
        with pytest.raises(T.TmdError) as e:
            T.tmd_decode(ctx, T.make_compressed(dev), out, T.TMD_VALIDATE, torch.cuda.current_stream().cuda_stream)
        assert e.value.status == T.TMD_ERR_CORRUPT
    finally:
        T.tmd_destroy(ctx)


def test_unchecked_ieee_sequences_equal_the_intrinsics():
    # the decode kernel's division / square-root fast sequences (no per-operation range check) and its fused
    # floor-clamp-convert against __fdiv_rn / __fsqrt_rn / floorf + clamp: every sqrt argument of the accepted range,
    # 2^33 division operand pairs of the accepted ranges (+ edge grid), every pattern for the conversion
    from paper_2411_02206_b200 import tmd as T
    assert T.tmd_selftest_ieee(33) == (0, 0, 0)


def _gpu_encode_unattached(geo, un):
    """tmd_encode_unattached on numpy cluster records -> dict of numpy arrays (u_* and u_bin_count)."""
    import torch
    from paper_2411_02206_b200 import tmd as T
    from tmd_inputs.layout import COMPRESSED_FIELDS
    ctx = T.tmd_create(geo, BZ)
    try:
        n = len(un)
        d_un = torch.from_numpy(np.ascontiguousarray(un).view(np.int32).reshape(-1, 4).copy()).cuda()
        tdt = {"<u2": torch.int16, "i1": torch.int8, "u1": torch.uint8, "<u4": torch.int32}
        out = {k: torch.full((n if w == "n_unattached" else geo.n_bins,), -1, dtype=tdt[dt], device="cuda")
               for k, (dt, w) in COMPRESSED_FIELDS.items() if k.startswith("u_")}
        ws = torch.empty(T.tmd_encode_unattached_workspace_bytes(ctx, n), dtype=torch.uint8, device="cuda")
        T.tmd_encode_unattached(ctx, d_un, out, ws, torch.cuda.current_stream().cuda_stream)
        return {k: v.cpu().numpy().view(np.dtype(COMPRESSED_FIELDS[k][0])) for k, v in out.items()}
    finally:
        T.tmd_destroy(ctx)


def _assert_unattached_encoding_equals_oracle(geo, un):
    from tmd_inputs.layout import CLUSTER_DTYPE
    want = O.encode(geo, BZ, np.zeros(0, np.uint16), np.zeros(0, np.float32), np.zeros(0, CLUSTER_DTYPE), np.zeros(0, np.uint8), un)
    got = _gpu_encode_unattached(geo, un)
    for k, v in got.items():
        assert np.array_equal(v, getattr(want, k)), f"{k}: " + first_mismatch(v, getattr(want, k))


def test_gpu_unattached_encoder_matches_oracle_encoder(phys_case):
    # "unassigned clusters are sorted by coordinate position ... stored as differences relative to the preceding
    # cluster": the library's per-bin sort + differencing produces the oracle encoder's bytes
    name, geo, ev, comp = phys_case
    got = _gpu_encode_unattached(geo, ev.un)
    for k, v in got.items():
        assert np.array_equal(v, getattr(comp, k)), f"{k}: " + first_mismatch(v, getattr(comp, k))


def test_gpu_unattached_encoder_ties_skew_and_empty():
    from tmd_inputs.layout import CLUSTER_DTYPE
    geo = build_geometry(36)
    rng = np.random.default_rng(91)
    # (a) heavy ties: few distinct times / pads / charges, so that the order is decided deep in the tuple, with exact duplicates
    n = 400_000
    un = np.zeros(n, CLUSTER_DTYPE)
    b = rng.integers(0, 40, n)                                  # 40 bins of ~10 000 clusters: several tiles per bin
    un["sector"], un["row"] = b // 8, 17 + b % 8
    un["time"] = rng.integers(0, 50, n); un["pad"] = rng.integers(0, 3, n); un["qtot"] = rng.integers(0, 2, n)
    un["qmax"] = rng.integers(0, 2, n); un["sigpad"] = rng.integers(0, 2, n); un["sigtime"] = rng.integers(0, 2, n)
    un["flags"] = rng.integers(0, 3, n)
    _assert_unattached_encoding_equals_oracle(geo, un)
    # (b) one bin far larger than a tile (eight merge passes), extreme values (the all-ones record equals the tile padding key)
    n = 300_000
    un = np.zeros(n, CLUSTER_DTYPE)
    un["sector"], un["row"] = 35, 151
    un["time"] = rng.integers(0, 2 ** 32, n); un["pad"] = rng.integers(0, 65536, n); un["qtot"] = rng.integers(0, 65536, n)
    un["qmax"] = rng.integers(0, 65536, n); un["sigpad"] = rng.integers(0, 256, n); un["sigtime"] = rng.integers(0, 256, n)
    un["flags"] = rng.integers(0, 256, n)
    for f, v in (("time", 2 ** 32 - 1), ("pad", 65535), ("qtot", 65535), ("qmax", 65535), ("sigpad", 255), ("sigtime", 255), ("flags", 255)):
        un[f][:5] = v
    extra = np.zeros(3000, CLUSTER_DTYPE)
    extra["sector"], extra["row"] = rng.integers(0, 36, 3000), rng.integers(0, 152, 3000)
    extra["time"] = rng.integers(0, 1000, 3000)
    _assert_unattached_encoding_equals_oracle(geo, np.concatenate((un, extra)))
    # (c) nothing at all, and exactly one tile
    _assert_unattached_encoding_equals_oracle(geo, np.zeros(0, CLUSTER_DTYPE))
    one = np.zeros(2048, CLUSTER_DTYPE)
    one["time"] = rng.permutation(2048)
    _assert_unattached_encoding_equals_oracle(geo, one)
    # a cluster without an output bin is reported
    from paper_2411_02206_b200 import tmd as T
    bad = np.zeros(10, CLUSTER_DTYPE)
    bad["row"][3] = 200
    with pytest.raises(T.TmdError) as e:
        _gpu_encode_unattached(geo, bad)
    assert e.value.status == T.TMD_ERR_CORRUPT


# ------------------------------------------------------------------------------------------------ entropy stage (rANS) in front
def _gpu_entropy_decode(blob: np.ndarray):
    """tmd_entropy_decode of a TMDZ container -> (dict of device tensors, error word)."""
    import torch
    from paper_2411_02206_b200 import tmd as T
    from tmd_inputs.layout import COMPRESSED_FIELDS
    n_trk, n_att, n_un, n_bins, total = T.tmd_entropy_sizes(blob[:64])
    assert total == blob.size
    lens = {"n_tracks": n_trk, "n_attached": n_att, "n_residuals": n_att - n_trk, "n_unattached": n_un, "n_bins": n_bins}
    tdt = {"<u2": torch.int16, "i1": torch.int8, "u1": torch.uint8, "<u4": torch.int32}
    out = {k: torch.full((lens[w],), -86, dtype=tdt[dt], device="cuda") for k, (dt, w) in COMPRESSED_FIELDS.items()}
    d_blob = torch.from_numpy(blob).cuda()
    d_err = torch.zeros(1, dtype=torch.int32, device="cuda")
    T.tmd_entropy_decode(blob[:T.ENTROPY_HEAD_BYTES], d_blob, out, d_err, torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    return out, int(d_err.item())


def _assert_arrays_equal(out: dict, comp):
    from tmd_inputs.layout import COMPRESSED_FIELDS
    for k, (dt, _) in COMPRESSED_FIELDS.items():
        got = out[k].cpu().numpy().view(np.dtype(dt))
        assert np.array_equal(got, getattr(comp, k)), f"{k}: " + first_mismatch(got, getattr(comp, k))


def test_entropy_decode_matches_oracle_and_feeds_the_decoder(phys_case):
    # PAPER.md L49 / L68: entropy decoding, then track-model decoding.  The container is written by the ORACLE encoder; the GPU
    # rANS decoder must restore every array of the compressed SoA bit for bit, and tmd_decode on those arrays (never leaving
    # the device) must give the oracle decoder's clusters.
    import torch
    from oracle import tmd_ans as ANS
    from paper_2411_02206_b200 import tmd as T
    from tmd_inputs.layout import CLUSTER_DTYPE
    name, geo, ev, comp = phys_case
    blob = ANS.encode_container(comp)
    out, err = _gpu_entropy_decode(blob)
    assert err == 0
    _assert_arrays_equal(out, comp)
    if name in ("c0", "c2_like"):
        ctx = T.tmd_create(geo, BZ)
        try:
            n = comp.n_attached + comp.n_unattached
            d_cl = torch.empty(n * 16, dtype=torch.uint8, device="cuda")
            d_bo = torch.empty(geo.n_bins + 1, dtype=torch.int32, device="cuda")
            ws = torch.empty(T.tmd_workspace_bytes(ctx, comp.n_tracks, comp.n_attached, comp.n_unattached), dtype=torch.uint8, device="cuda")
            T.tmd_decode(ctx, T.make_compressed(out), T.make_output(d_cl, d_bo, ws), 0, torch.cuda.current_stream().cuda_stream)
            torch.cuda.synchronize()
            want = O.decode(geo, BZ, comp)
            assert np.array_equal(d_bo.cpu().numpy().view(np.uint32), want[1])
            assert d_cl.cpu().numpy().view(CLUSTER_DTYPE).tobytes() == want[0].tobytes()
        finally:
            T.tmd_destroy(ctx)


def test_entropy_decode_edge_cases_and_library_encoder():
    from oracle import tmd_ans as ANS
    from paper_2411_02206_b200 import tmd as T
    from tmd_inputs.layout import COMPRESSED_FIELDS
    geo = build_geometry(36)
    cases = [random_compressed(geo, 3000, 40_000, 101, max_ncl=120),          # several 64 KiB chunks per array, ragged tails
             random_compressed(geo, 1, 0, 102), random_compressed(geo, 0, 7, 103), Compressed.empty(0, 0, 0, geo.n_bins),
             degenerate_same_bin(geo, np.full(400, 300, np.uint16), 104, n_un=50_001)]   # planes with one symbol only
    for i, c in enumerate(cases):
        for blob in (ANS.encode_container(c), T.tmd_entropy_encode_host({k: np.ascontiguousarray(getattr(c, k)) for k in COMPRESSED_FIELDS}, geo.n_bins)):
            out, err = _gpu_entropy_decode(blob)
            assert err == 0, i
            _assert_arrays_equal(out, c)
    # corrupt containers are reported, not followed out of bounds: a table that does not sum to 4096, a block table of garbage
    c = cases[0]
    blob = ANS.encode_container(c)
    rec = blob[64:96]
    t_off, b_off = int(rec[16:24].view(np.uint64)[0]), int(rec[24:32].view(np.uint64)[0])
    bad = blob.copy(); bad[t_off:t_off + 2].view(np.uint16)[0] += 1
    assert _gpu_entropy_decode(bad)[1] & 1
    bad = blob.copy(); bad[b_off:b_off + 8].view(np.uint32)[:] = (0xFFFFFF00, 5)
    assert _gpu_entropy_decode(bad)[1] & 4
    # a block position that is in order and in bounds but not 4-byte aligned (its 32 states are read as words): reported,
    # not followed into a misaligned-address fault that would poison the CUDA context for every later test
    starts = blob[b_off:b_off + 8].view(np.uint32)
    for shift in (1, 2, 3):
        bad = blob.copy(); bad[b_off:b_off + 4].view(np.uint32)[0] = starts[0] + shift
        assert _gpu_entropy_decode(bad)[1] & 4, shift
    # bit flips inside a block: one of its words, one of its coder states
    s0, s1 = int(starts[0]), int(starts[1])
    assert s1 - s0 > 4 * 32 + 64
    bad = blob.copy(); bad[s0 + 4 * 32 + 40] ^= 0x10
    assert _gpu_entropy_decode(bad)[1] & (8 | 2)
    bad = blob.copy(); bad[s0 + 4 * 7 + 1] ^= 0x01
    assert _gpu_entropy_decode(bad)[1] & (8 | 2)
    # a plane directory that points far outside the container (offsets near 2^64 must not wrap the host's range check)
    for field in (16, 24):
        for v in (0xFFFFFFFFFFFFFF00, 0xFFFFFFFFFFFFFFFC, blob.size, blob.size - 4):
            bad = blob.copy(); bad[64 + field:64 + field + 8].view(np.uint64)[0] = v
            with pytest.raises(T.TmdError) as e:
                _gpu_entropy_decode(bad)
            assert e.value.status == T.TMD_ERR_CORRUPT, (field, hex(v))
    out, err = _gpu_entropy_decode(blob)                    # the context survived all of the above
    assert err == 0
    _assert_arrays_equal(out, c)


def test_container_host_entry_point_matches_oracle(phys_case):
    # The deployment shape: a TMDZ container in host memory in, clusters in host memory out, through
    # tmd_decode_container_host_async.  The container is written by the ORACLE (oracle encoder -> oracle rANS coder) and the
    # result must be orc_decode's, record for record.  Frames alternate between the two pipeline slots, mixed with the
    # array-input entry point on the other slot.
    import torch
    from oracle import tmd_ans as ANS
    from paper_2411_02206_b200 import tmd as T
    from tmd_inputs.layout import CLUSTER_DTYPE, COMPRESSED_FIELDS
    from gpu_util import _as_torch
    name, geo, ev, comp = phys_case
    blob = torch.from_numpy(ANS.encode_container(comp)).pin_memory()
    want_cl, want_bo, _ = O.decode(geo, BZ, comp)
    n = comp.n_attached + comp.n_unattached
    assert T.tmd_entropy_sizes(blob.numpy()[:64])[:3] == (comp.n_tracks, comp.n_attached, comp.n_unattached)
    ctx = T.tmd_create(geo, BZ)
    try:
        outs = [(torch.full((n * 16,), 0xEE, dtype=torch.uint8).pin_memory(), torch.zeros(geo.n_bins + 1, dtype=torch.int32).pin_memory())
                for _ in range(3)]
        h_in = {k: _as_torch(np.ascontiguousarray(getattr(comp, k))).pin_memory() for k in COMPRESSED_FIELDS}
        T.tmd_decode_container_host_async(ctx, blob, T.make_output(*outs[0]), 0, 0)
        T.tmd_decode_host_async(ctx, T.make_compressed(h_in), T.make_output(*outs[1]), 0, 1)       # arrays in, other slot
        T.tmd_decode_container_host_async(ctx, blob, T.make_output(*outs[2]), 0, 0)               # waits for slot 0's first frame
        for s_ in range(T.TMD_HOST_SLOTS):
            T.tmd_host_wait(ctx, s_)
        for hc, hb in outs:
            assert np.array_equal(hb.numpy().view(np.uint32), want_bo)
            assert hc.numpy().view(CLUSTER_DTYPE).tobytes() == want_cl.tobytes()
        if name == "c0":
            # a damaged container is reported by tmd_host_wait; a container of another geometry, a non-container and the
            # synchronising flag are refused at the call
            bad = blob.clone()
            rec = bad.numpy()[64:96]
            b_off = int(rec[24:32].view(np.uint64)[0])
            s0 = int(bad.numpy()[b_off:b_off + 4].view(np.uint32)[0])
            bad.numpy()[s0 + 4 * 32 + 10] ^= 0x04
            bad = bad.pin_memory()
            T.tmd_decode_container_host_async(ctx, bad, T.make_output(*outs[0]), 0, 1)
            with pytest.raises(T.TmdError) as e:
                T.tmd_host_wait(ctx, 1)
            assert e.value.status == T.TMD_ERR_CORRUPT
            T.tmd_decode_container_host_async(ctx, blob, T.make_output(*outs[0]), 0, 1)          # the slot is usable again
            T.tmd_host_wait(ctx, 1)
            assert outs[0][0].numpy().view(CLUSTER_DTYPE).tobytes() == want_cl.tobytes()
            with pytest.raises(T.TmdError) as e:
                T.tmd_decode_container_host_async(ctx, blob, T.make_output(*outs[0]), T.TMD_VALIDATE, 0)
            assert e.value.status == T.TMD_ERR_ARG
            junk = torch.zeros(4096, dtype=torch.uint8).pin_memory()
            with pytest.raises(T.TmdError) as e:
                T.tmd_decode_container_host_async(ctx, junk, T.make_output(*outs[0]), 0, 0)
            assert e.value.status == T.TMD_ERR_CORRUPT
            other = T.tmd_create(build_geometry(36 if geo.n_sectors_out == 2 else 2), BZ)
            try:
                with pytest.raises(T.TmdError) as e:
                    T.tmd_decode_container_host_async(other, blob, T.make_output(*outs[0]), 0, 0)
                assert e.value.status == T.TMD_ERR_ARG
            finally:
                T.tmd_destroy(other)
    finally:
        T.tmd_destroy(ctx)
