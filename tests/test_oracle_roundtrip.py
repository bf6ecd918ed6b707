"""decode(encode(x)) == x and structural invariants of the oracle codec.

x = cluster truth from tmd_inputs.physical (float64 helices, no codec arithmetic); the expected decoder output is
`canonical(x)`, built with numpy library sorts only.  PAPER.md L68: decoding must "restore the original values".
"""
import numpy as np
import pytest

from oracle import tmd_oracle as O
from tmd_inputs import build_geometry, physical as ph

BZ = 0.5

CASES = {
    "c0": (lambda: ph.config0(), 2),
    "c1": (lambda: ph.config1(), 36),
    "c2_like": (lambda: ph.config2_like(4000, 60_000), 36),
    "c4_like": (lambda: ph.config4_like(20_000, 50_000), 36),
}


@pytest.fixture(scope="module", params=list(CASES))
def case(request):
    mk, nsec = CASES[request.param]
    geo = build_geometry(nsec)
    ev = ph.generate_event(mk(), geo)
    comp = O.encode(geo, BZ, ev.trk_ncl, ev.trk_qptf, ev.att, ev.leg, ev.un)
    return request.param, geo, ev, comp


def test_round_trip_is_byte_exact(case):
    name, geo, ev, comp = case
    cl, bo, _ = O.decode(geo, BZ, comp)
    want, want_bo = ph.canonical(ev, geo)
    assert np.array_equal(bo, want_bo)
    assert cl.tobytes() == want.tobytes()


def test_shape_of_the_workload(case):
    name, geo, ev, comp = case
    comp.check_shapes()
    ncl = ev.trk_ncl.astype(np.int64)
    if name == "c0":        # BASELINE.json config 0
        assert len(ncl) == 200 and 20 <= ncl.min() and ncl.max() <= 152 and comp.n_unattached == 5000
        assert set(np.unique(ev.att["sector"])) <= {0, 1}
    if name == "c1":        # config 1: 10k tracks, ~1.2M attached, 300k unattached, ~10% loopers with 2-3 legs
        assert len(ncl) == 10_000 and 1.1e6 < ncl.sum() < 1.35e6 and comp.n_unattached == 300_000
        assert ev.leg.max() >= 2 and (comp.a_secleg & 0x3F != 0).sum() > 5000
    if name == "c4_like":   # config 4 shape: short tracks, mean ~40, a few long multi-leg loopers
        assert 25 < ncl.mean() < 50 and ncl.max() > 400 and ncl.min() == 1


def test_invariants(case):
    name, geo, ev, comp = case
    cl, bo, _ = O.decode(geo, BZ, comp)
    n_bins = geo.n_bins
    # per-bin counts conserved: bin_offset[b+1]-bin_offset[b] == att_cnt[b] + u_bin_count[b]; total conserved
    abin = ev.att["sector"].astype(np.int64) * geo.n_rows + ev.att["row"]
    att_cnt = np.bincount(abin, minlength=n_bins)
    assert np.array_equal(np.diff(bo.astype(np.int64)), att_cnt + comp.u_bin_count)
    assert int(bo[-1]) == comp.n_attached + comp.n_unattached
    # every record sits in its own bin's range
    obin = cl["sector"].astype(np.int64) * geo.n_rows + cl["row"]
    assert np.array_equal(obin, np.repeat(np.arange(n_bins), np.diff(bo.astype(np.int64))))
    assert np.all(cl["zero"] == 0)
    # every attached cluster's row lies inside its track's generated row range
    off = np.concatenate(([0], np.cumsum(ev.trk_ncl.astype(np.int64))))
    lo = np.minimum.reduceat(ev.att["row"], off[:-1]); hi = np.maximum.reduceat(ev.att["row"], off[:-1])
    t_of = np.repeat(np.arange(len(ev.trk_ncl)), ev.trk_ncl)
    assert np.all((ev.att["row"] >= lo[t_of]) & (ev.att["row"] <= hi[t_of]))
    # stored streams respect the format (C2): rowdiff < n_rows, sector step < n_az, bit 6 clear, |qpt| <= 127
    assert comp.a_rowdiff.max(initial=0) < geo.n_rows
    assert np.all((comp.a_secleg & 0x3F) < geo.n_az) and np.all((comp.a_secleg & 0x40) == 0)
    assert np.all(np.abs(comp.trk_qpt.astype(np.int64)) <= 127)
    # unattached clusters are stored sorted by time inside each bin => time differences never wrap
    ustart = np.concatenate(([0], np.cumsum(comp.u_bin_count.astype(np.int64))))
    first = np.zeros(comp.n_unattached, bool); first[ustart[:-1][comp.u_bin_count > 0]] = True
    un_sorted_time = np.cumsum(np.where(first, 0, comp.u_timediff.astype(np.int64)))
    assert np.all(comp.u_timediff.astype(np.int64)[~first] < 2 ** 31)
    assert len(un_sorted_time) == comp.n_unattached


def test_realistic_residuals_are_small(case):
    # with sigma = 0.05 cm noise the residuals are a few codes (SURVEY C3 "scratch check": median <= 12 codes)
    name, geo, ev, comp = case
    pr = np.abs(comp.a_padres.astype(np.int16).astype(np.int64))
    tr = np.abs(comp.a_timeres.astype(np.int32).astype(np.int64))
    assert np.median(pr) <= 12 and np.median(tr) <= 12


def test_encoder_is_order_independent_for_unattached(case):
    name, geo, ev, comp = case
    rng = np.random.default_rng(0)
    un2 = ev.un[rng.permutation(len(ev.un))]
    comp2 = O.encode(geo, BZ, ev.trk_ncl, ev.trk_qptf, ev.att, ev.leg, un2)
    for k in ("u_paddiff", "u_timediff", "u_qtot", "u_qmax", "u_flags", "u_sigpad", "u_sigtime", "u_bin_count"):
        assert np.array_equal(getattr(comp, k), getattr(comp2, k)), k
