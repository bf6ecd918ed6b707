"""Pins for the CPU oracle (oracle/tmd_oracle.c) against things other than itself.

The paper prints no worked example and no formula, so the pins are:
  * the worked trace of SURVEY.md §8(c)-C9 (tests/golden/c9_trace.txt), bit for bit;
  * geometric closed forms evaluated here in float64 (straight line / exact circle through the beam line);
  * physical fidelity: noiseless exact helices (tmd_inputs.physical, float64) must leave residuals of a few codes;
  * library routines: numpy.cumsum for offsets and unattached sums, numpy stable argsort for the canonical order;
  * the C8 hand example for the unattached decoder; brute-force assembly on small inputs.
"""
import os

import numpy as np
import pytest

from conftest import parse_golden_trace, residual_meta
from oracle import tmd_oracle as O
from tmd_inputs import build_geometry, physical as ph
from tmd_inputs.adversarial import random_compressed
from tmd_inputs.layout import CLUSTER_DTYPE, Compressed

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "c9_trace.txt")
BZ = 0.5


def f32(bits):
    return np.array([bits], np.uint32).view(np.float32)[0]


# ---------------------------------------------------------------------------------------------- geometry (C1)
def test_geometry_pins(geo36):
    # SURVEY.md §8(c)-C1 "Pins"
    assert [int(geo36.row_npads[r]) for r in (0, 62, 63, 96, 97, 126, 127, 151)] == [74, 114, 78, 98, 100, 120, 122, 144]
    assert int(geo36.row_npads.sum()) == 15556
    bits = lambda a, i: int(a[i:i + 1].view(np.uint32)[0])
    assert bits(geo36.row_x, 98) == 0x432C3333 and bits(geo36.row_x, 151) == 0x43750000
    assert bits(geo36.row_padw, 0) == 0x3ECCCCCD
    assert bits(geo36.row_inv_padw, 0) == 0x40200000 and bits(geo36.row_inv_padw, 100) == 0x3FD55555
    assert int(np.array([geo36.cos_a]).view(np.uint32)[0]) == 0x3F708FB2
    assert int(np.array([geo36.sin_a]).view(np.uint32)[0]) == 0x3EAF1D44
    assert np.all(geo36.row_npads % 2 == 0) and np.all(np.diff(geo36.row_x) > 0)


# ---------------------------------------------------------------------------------------------- worked trace (C9)
def test_c9_worked_trace_bit_exact(geo36):
    gold = parse_golden_trace(GOLDEN)
    sec0, row0, P0, T0, qpt, ncl = gold["track"]
    res = np.array(gold["res"], dtype=np.int64)
    assert len(res) == ncl - 1
    r = O.decode_track(geo36, BZ, qpt, sec0, row0, P0, T0, res[:, 0], res[:, 1], res[:, 2], res[:, 3],
                       want_trace=True, probe_step=0)
    assert [int(v) for v in r["probe"]] == gold["init"]          # x y u sp dt k after C3-1, C3-2
    cols = ("sec", "row", "dir", "ok", "x", "y", "sp", "sp2", "y2", "u2", "s", "P_pred", "T_pred", "P", "T",
            "yn", "un", "spn", "dtn", "kn")
    for step, tr in zip(gold["steps"], r["trace"]):
        j, want = step[0], step[1:]
        got = [getattr(tr, c) for c in cols]
        for c, g, w in zip(cols, got, want):
            assert g == w, f"cluster j={j} column {c}: oracle {g:#x} golden {w:#x}"
    got_out = list(zip(r["sec"].tolist(), r["row"].tolist(), r["P"].tolist(), r["T"].tolist()))
    assert got_out == [tuple(o) for o in gold["out"]]


def test_probe_steps_follow_trace(geo36):
    gold = parse_golden_trace(GOLDEN)
    sec0, row0, P0, T0, qpt, ncl = gold["track"]
    res = np.array(gold["res"], dtype=np.int64)
    for step in (1, 3, ncl - 1, 10 ** 6):        # probe_step > ncl-1 clamps to the final state
        r = O.decode_track(geo36, BZ, qpt, sec0, row0, P0, T0, res[:, 0], res[:, 1], res[:, 2], res[:, 3],
                           want_trace=True, probe_step=step)
        tr = r["trace"][min(step, ncl - 1) - 1]
        want_x = int(geo36.row_x[tr.row:tr.row + 1].view(np.uint32)[0])     # C3-9: "always x = xt"
        assert [int(v) for v in r["probe"]] == [want_x, tr.yn, tr.un, tr.spn, tr.dtn, tr.kn]


# ---------------------------------------------------------------------------------------------- closed forms
@pytest.mark.parametrize("row0", [0, 62, 96])
def test_closed_form_radial_track(geo36, row0):
    # qpt=0, y0=0, residuals 0, rowdiff 1 => sp=0, dy=0, P = 32*npads(row), T = T0 on every row
    n = 152 - row0
    z = np.zeros(n - 1, np.int64)
    r = O.decode_track(geo36, BZ, 0, 5, row0, 32 * int(geo36.row_npads[row0]), 123456, z + 1, z, z, z, want_trace=True)
    rows = np.arange(row0, 152)
    assert np.array_equal(r["row"], rows) and np.all(r["sec"] == 5)
    assert np.array_equal(r["P"], 32 * geo36.row_npads[rows].astype(np.int64))
    assert np.all(r["T"] == 123456)
    for tr in r["trace"]:
        assert tr.ok == 1 and tr.P == tr.P_pred and tr.T == tr.T_pred and f32(tr.spn) == 0.0 and f32(tr.dtn) == 0.0


def test_closed_form_first_step_on_exact_circle(geo36):
    # One propagation step from the first cluster, zero residual: the rebuilt pad is the model's prediction, which
    # must be the exact circle of curvature kappa = qpt/16 * 0.00299792458*Bz through the beam line and the first
    # cluster (C3-2 start direction, C3-6 chord identity), rounded to a code.  Circle evaluated here in float64.
    # (Only ONE step is a closed form: with zero residuals the filter feeds its own rounding back and locks onto an
    # integer code increment per row, so longer zero-residual tracks drift off the circle by design.)
    x = geo36.row_x_f64; w = geo36.row_padw_f64; half = geo36.row_npads / 2.0
    worst = 0.0
    n = 0
    for qpt in (-100, -60, -20, 0, 20, 60, 100):
        kappa = qpt / 16.0 * 0.00299792458 * BZ
        for row0 in range(0, 150, 7):
            for rd in (1, 2, 5):
                row1 = row0 + rd
                if row1 > 151:
                    continue
                for padfrac in (0.1, 0.37, 0.5, 0.81):
                    P0 = int(padfrac * geo36.row_npads[row0] * 64)
                    y0 = (P0 / 64.0 - half[row0]) * w[row0]
                    L = np.hypot(x[row0], y0)
                    if abs(kappa * L / 2.0) >= 1:
                        continue
                    phi_org = np.arctan2(y0, x[row0]) - np.arcsin(kappa * L / 2.0)     # direction at the beam line
                    S0, S1 = np.sin(phi_org) + kappa * x[row0], np.sin(phi_org) + kappa * x[row1]
                    if abs(S1) > 0.9:
                        continue
                    y1 = y0 + (x[row1] - x[row0]) * (S0 + S1) / (np.sqrt(1 - S0 * S0) + np.sqrt(1 - S1 * S1))
                    want = (y1 / w[row1] + half[row1]) * 64
                    if not (0 <= want <= 65535):
                        continue
                    r = O.decode_track(geo36, BZ, qpt, 0, row0, P0, 5000, [rd], [0], [0], [0])
                    worst = max(worst, abs(float(r["P"][1]) - want)); n += 1
                    assert r["row"][1] == row1 and r["T"][1] == 5000
    assert n > 1500
    assert worst <= 0.5 + 0.02, worst          # round-to-nearest code + fp32 noise


def test_sector_rotation_matches_float64_geometry(geo36):
    # One step that changes sector by +1 (d=1) or -1 (d=17) and jumps `rd` rows, zero residual: the rebuilt pad must be
    # the exact circle, expressed in the neighbouring sector's frame (rotation by -/+20 deg), rounded to a code.
    # Pins the signs and the operand order of C3-5.  Float64 geometry evaluated here.
    x = geo36.row_x_f64; w = geo36.row_padw_f64; half = geo36.row_npads / 2.0
    a20 = np.deg2rad(20.0)
    n = {1: 0, 17: 0}
    worst = 0.0
    for d, sgn in ((1, +1.0), (17, -1.0)):
        for qpt in (sgn * 60, sgn * 90, sgn * 120):
            kappa = qpt / 16.0 * 0.00299792458 * BZ
            for row0 in range(0, 130, 5):
                for rd in (8, 14, 20):
                    row1 = row0 + rd
                    if row1 > 151:
                        continue
                    for edge in (0.90, 0.97):                      # start near the edge the track is bending towards
                        P0 = int((0.5 + sgn * 0.5 * edge) * geo36.row_npads[row0] * 64)
                        y0 = (P0 / 64.0 - half[row0]) * w[row0]
                        L = np.hypot(x[row0], y0)
                        if abs(kappa * L / 2.0) >= 0.9:
                            continue
                        phi_s = np.arctan2(y0, x[row0]) + np.arcsin(kappa * L / 2.0)      # local direction at cluster 0
                        xr = x[row0] * np.cos(a20) + sgn * y0 * np.sin(a20)               # same point, neighbour frame
                        yr = y0 * np.cos(a20) - sgn * x[row0] * np.sin(a20)
                        S0 = np.sin(phi_s - sgn * a20)
                        S1 = S0 + kappa * (x[row1] - xr)
                        if abs(np.sin(phi_s)) > 0.9 or abs(S0) > 0.9 or abs(S1) > 0.9:    # stay clear of the SP_MAX clamp
                            continue
                        y1 = yr + (x[row1] - xr) * (S0 + S1) / (np.sqrt(1 - S0 * S0) + np.sqrt(1 - S1 * S1))
                        want = (y1 / w[row1] + half[row1]) * 64
                        if not (0 <= want < geo36.row_npads[row1] * 64):
                            continue
                        r = O.decode_track(geo36, BZ, int(qpt), 4, row0, P0, 9000, [rd], [d], [0], [0])
                        assert r["sec"][1] == (5 if d == 1 else 3) and r["row"][1] == row1
                        worst = max(worst, abs(float(r["P"][1]) - want)); n[d] += 1
    assert n[1] > 20 and n[17] > 20, n
    assert worst <= 0.5 + 0.05, worst
    # the side is kept: az wraps inside side C (sector 18+17 -> 18) and inside side A (sector 0, d=17 -> 17)
    assert O.decode_track(geo36, BZ, 0, 35, 40, 3000, 9000, [1], [0x01], [0], [0])["sec"][1] == 18
    assert O.decode_track(geo36, BZ, 0, 0, 40, 3000, 9000, [1], [17], [0], [0])["sec"][1] == 17


# ---------------------------------------------------------------------------------------------- physical fidelity
@pytest.mark.parametrize("seed", [11, 12])
def test_noiseless_helices_leave_tiny_residuals(geo36, seed):
    # Exact float64 helices (no noise) through the oracle ENCODER: if the model (C3) dropped a term, had a sign or an
    # index wrong, or rotated/mirrored the wrong way, the residuals would be tens to thousands of codes.
    cfg = ph.config1(3000, 100, seed=seed)
    cfg.noise_cm = 0.0; cfg.looper_frac = 0.3; cfg.looper_pt = (0.13, 0.18)     # |qpt| < 127: no curvature clamp
    ev = ph.generate_event(cfg, geo36)
    comp = O.encode(geo36, BZ, ev.trk_ncl, ev.trk_qptf, ev.att, ev.leg, ev.un)
    pr = np.abs(comp.a_padres.astype(np.int16).astype(np.int64))
    tr = np.abs(comp.a_timeres.astype(np.int32).astype(np.int64))
    tt, jj, leg, since = residual_meta(ev)
    unclamped = (np.abs(comp.trk_qpt.astype(int)) < 127)[tt]
    secchg = (comp.a_secleg & 0x3F) != 0
    sel = (leg == 0) & (jj >= 10) & unclamped
    assert sel.sum() > 250_000
    assert np.percentile(pr[sel], 99) <= 2 and np.percentile(tr[sel], 99) <= 3 and pr[sel].max() <= 40
    sel2 = sel & secchg                                    # straight after a sector rotation
    assert sel2.sum() > 3000 and np.percentile(pr[sel2], 99) <= 16 and np.percentile(tr[sel2], 99) <= 10
    sel3 = (leg == 1) & (since >= 25) & unclamped          # return leg of a looper, once the filter has re-converged
    assert sel3.sum() > 10_000 and np.percentile(pr[sel3], 99) <= 2 and np.percentile(tr[sel3], 99) <= 2


# ---------------------------------------------------------------------------------------------- unattached (C4)
def _empty_attached(n_bins, counts, paddiff, timediff, rng=None):
    n = int(np.sum(counts))
    c = Compressed.empty(0, 0, n, n_bins)
    c.u_bin_count[:] = counts
    c.u_paddiff[:] = np.asarray(paddiff, np.int64) & 0xFFFF
    c.u_timediff[:] = np.asarray(timediff, np.int64) & 0xFFFFFFFF
    if rng is not None:
        c.u_qtot[:] = rng.integers(0, 65536, n); c.u_qmax[:] = rng.integers(0, 65536, n)
        c.u_flags[:] = rng.integers(0, 256, n); c.u_sigpad[:] = rng.integers(0, 256, n); c.u_sigtime[:] = rng.integers(0, 256, n)
    return c


def test_unattached_hand_example(geo36):
    # SURVEY C8 hand example
    counts = np.zeros(geo36.n_bins, np.uint32); counts[:3] = [3, 0, 2]
    c = _empty_attached(geo36.n_bins, counts, [100, 65530, 7, 50, 3], [1000, 5, 0, 20, 4294967295])
    cl, bo, _ = O.decode(geo36, BZ, c)
    assert cl["pad"].tolist() == [100, 94, 101, 50, 53]
    assert cl["time"].tolist() == [1000, 1005, 1005, 20, 19]
    assert cl["row"].tolist() == [0, 0, 0, 2, 2] and cl["sector"].tolist() == [0] * 5
    assert bo[:4].tolist() == [0, 3, 3, 5] and bo[-1] == 5


def test_unattached_equals_numpy_cumsum(geo36):
    rng = np.random.default_rng(5)
    counts = rng.poisson(3.0, geo36.n_bins).astype(np.uint32)
    counts[rng.integers(0, geo36.n_bins, 50)] = 0
    counts[7] = 3000
    n = int(counts.sum())
    c = _empty_attached(geo36.n_bins, counts, rng.integers(0, 65536, n), rng.integers(0, 2 ** 32, n), rng)
    cl, bo, _ = O.decode(geo36, BZ, c)
    starts = np.concatenate(([0], np.cumsum(counts.astype(np.int64))))
    assert np.array_equal(bo, starts.astype(np.uint32))
    for b in np.nonzero(counts)[0]:
        s, e = starts[b], starts[b + 1]
        assert np.array_equal(cl["pad"][s:e], np.cumsum(c.u_paddiff[s:e], dtype=np.uint16))
        assert np.array_equal(cl["time"][s:e], np.cumsum(c.u_timediff[s:e], dtype=np.uint32))
        assert np.all(cl["sector"][s:e] == b // 152) and np.all(cl["row"][s:e] == b % 152)
    for f, g in (("qtot", "u_qtot"), ("qmax", "u_qmax"), ("flags", "u_flags"), ("sigpad", "u_sigpad"), ("sigtime", "u_sigtime")):
        assert np.array_equal(cl[f], getattr(c, g))
    assert np.all(cl["zero"] == 0)


# ---------------------------------------------------------------------------------------------- assembly (A1, A3-A6, C5)
def brute_force_decode(geo, c):
    """Per-track decode with slices cut by numpy.cumsum, canonical order by numpy stable argsort."""
    ncl = c.trk_ncl.astype(np.int64)
    off = np.concatenate(([0], np.cumsum(ncl)))          # A1: exclusive prefix sum (library routine)
    sec = np.zeros(c.n_attached, np.int64); row = np.zeros_like(sec); P = np.zeros_like(sec); T = np.zeros_like(sec)
    for t in range(c.n_tracks):
        r0 = off[t] - t                                   # roff[t]
        n = ncl[t] - 1
        r = O.decode_track(geo, BZ, int(c.trk_qpt[t]), int(c.trk_sec0[t]), int(c.trk_row0[t]), int(c.trk_pad0[t]),
                           int(c.trk_time0[t]), c.a_rowdiff[r0:r0 + n], c.a_secleg[r0:r0 + n],
                           c.a_padres[r0:r0 + n], c.a_timeres[r0:r0 + n])
        s = slice(off[t], off[t + 1])
        sec[s], row[s], P[s], T[s] = r["sec"], r["row"], r["P"], r["T"]
    att = np.zeros(c.n_attached, CLUSTER_DTYPE)
    att["sector"], att["row"], att["pad"], att["time"] = sec, row, P, T
    att["qtot"], att["qmax"], att["flags"], att["sigpad"], att["sigtime"] = c.a_qtot, c.a_qmax, c.a_flags, c.a_sigpad, c.a_sigtime
    abin = sec * geo.n_rows + row
    a_cnt = np.bincount(abin, minlength=geo.n_bins)
    att_sorted = att[np.argsort(abin, kind="stable")]     # C5: stable sort of the g-ordered stream by bin
    un = np.zeros(c.n_unattached, CLUSTER_DTYPE)
    ustart = np.concatenate(([0], np.cumsum(c.u_bin_count.astype(np.int64))))
    for b in np.nonzero(c.u_bin_count)[0]:
        s = slice(ustart[b], ustart[b + 1])
        un["pad"][s] = np.cumsum(c.u_paddiff[s], dtype=np.uint16); un["time"][s] = np.cumsum(c.u_timediff[s], dtype=np.uint32)
        un["sector"][s] = b // geo.n_rows; un["row"][s] = b % geo.n_rows
    un["qtot"], un["qmax"], un["flags"], un["sigpad"], un["sigtime"] = c.u_qtot, c.u_qmax, c.u_flags, c.u_sigpad, c.u_sigtime
    bo = np.concatenate(([0], np.cumsum(a_cnt + c.u_bin_count))).astype(np.uint32)
    out = np.zeros(c.n_attached + c.n_unattached, CLUSTER_DTYPE)
    astart = np.concatenate(([0], np.cumsum(a_cnt)))
    for b in range(geo.n_bins):
        out[bo[b]: bo[b] + a_cnt[b]] = att_sorted[astart[b]:astart[b + 1]]
        out[bo[b] + a_cnt[b]: bo[b + 1]] = un[ustart[b]:ustart[b + 1]]
    return out, bo


@pytest.mark.parametrize("seed,n_tracks,n_un", [(1, 300, 4000), (2, 1, 0), (3, 50, 0), (4, 0, 100)])
def test_full_decode_equals_brute_force_assembly(geo36, seed, n_tracks, n_un):
    c = random_compressed(geo36, n_tracks, n_un, seed)
    cl, bo, _ = O.decode(geo36, BZ, c)
    want, want_bo = brute_force_decode(geo36, c)
    assert np.array_equal(bo, want_bo)
    assert cl.tobytes() == want.tobytes()


def test_empty_input(geo36):
    c = Compressed.empty(0, 0, 0, geo36.n_bins)
    cl, bo, _ = O.decode(geo36, BZ, c)
    assert len(cl) == 0 and np.all(bo == 0)


def test_corrupt_counts_rejected(geo36):
    c = random_compressed(geo36, 10, 10, 9)
    c.u_bin_count[0] += 1
    with pytest.raises(RuntimeError):
        O.decode(geo36, BZ, c)
    c = random_compressed(geo36, 10, 10, 9)
    c.trk_ncl[3] = 0
    with pytest.raises(RuntimeError):
        O.decode(geo36, BZ, c)
