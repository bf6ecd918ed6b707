"""Pins the oracle's track model (oracle/tmd_oracle.c: orc_init, orc_step) to a SECOND, independent evaluation of the op
list SURVEY.md §8(c)-C3: tests/c3_numpy.py (numpy float32 scalars, written from the survey text, shares nothing with
oracle/).  Every column of the per-step trace (SURVEY C9's 20 columns) and the initial / final state are compared bit for
bit (NaN compares equal to NaN, reading 15), on

  (a) every track of BASELINE.json config 0 (physical helices through the oracle ENCODER),
  (b) crafted tracks that force the branches no round-trip or physical input reaches: several consecutive `ok = 0` steps
      (C3-7 / C3-9, reading 8), multi-step sector rotations in both directions (C3-5), `dt` saturating at +-DT_MAX,
      `T_pred` at 2^24-1, `P_pred` at 65535 and 0, the start-direction clamp of C3-2, out-of-format bytes (reading 19:
      rowdiff in [152, 255] on an inward leg, sector steps in [18, 63], bit 6 of a_secleg),
  (c) 1000 tracks of random bytes.

Why this exists: encoder and decoder share orc_step, so `decode(encode(x)) == x` is blind to a mistake in it; the C9 trace
has `ok = 1` on every row.  The table "mutation -> failing test" is in DESIGN.md §4.
PAPER.md L70: "propagates it through the TPC ... using the residuals given in input and the reconstructed track".
"""
import numpy as np
import pytest

from c3_numpy import COLUMNS, FLOAT_COLUMNS, ONLY_IF_OK, Model, same_bits
from oracle import tmd_oracle as O
from tmd_inputs import physical as ph
from tmd_inputs.adversarial import random_compressed

BZ = 0.5


def compare_track(geo, model, qpt, sec0, row0, P0, T0, rowdiff, secleg, padres, timeres, tag=""):
    """Oracle (C) vs the independent numpy evaluation: outputs, every trace column, initial and final state.  Returns the trace."""
    rowdiff = np.asarray(rowdiff, np.int64); secleg = np.asarray(secleg, np.int64)
    padres = np.asarray(padres, np.int64); timeres = np.asarray(timeres, np.int64)
    got = O.decode_track(geo, BZ, qpt, sec0, row0, P0, T0, rowdiff, secleg, padres, timeres, want_trace=len(rowdiff) > 0,
                         probe_step=0)
    want = model.decode_track(qpt, sec0, row0, P0, T0, rowdiff, secleg, padres, timeres)
    for c, w in zip(("x", "y", "u", "sp", "dt", "k"), want["init"]):
        g = int(got["probe"][("x", "y", "u", "sp", "dt", "k").index(c)])
        assert same_bits(g, w), f"{tag} init {c}: oracle {g:#010x} independent {w:#010x}"
    for key in ("sec", "row", "P", "T"):
        assert got[key].tolist() == want[key], f"{tag} rebuilt {key}"
    for j, (tg, tw) in enumerate(zip(got.get("trace", []), want["trace"]), start=1):
        for c in COLUMNS:
            g, w = getattr(tg, c), tw[c]
            if c in ONLY_IF_OK and not tw["ok"]:
                continue
            same = same_bits(g, w) if c in FLOAT_COLUMNS else g == w
            assert same, f"{tag} cluster j={j} column {c}: oracle {g:#x} independent {w:#x}"
    fin = O.decode_track(geo, BZ, qpt, sec0, row0, P0, T0, rowdiff, secleg, padres, timeres, probe_step=0xFFFFFFFF)["probe"]
    for c, g, w in zip(("x", "y", "u", "sp", "dt", "k"), fin.tolist(), want["final"]):
        assert same_bits(int(g), w), f"{tag} final {c}: oracle {int(g):#010x} independent {w:#010x}"
    return want["trace"]


def f32(b):
    return float(np.array([b], np.uint32).view(np.float32)[0])


# ---------------------------------------------------------------------------------------------- (a) config 0, every track
def test_config0_every_track_every_step(geo2):
    ev = ph.generate_event(ph.config0(), geo2)
    comp = O.encode(geo2, BZ, ev.trk_ncl, ev.trk_qptf, ev.att, ev.leg, ev.un)
    model = Model(geo2, BZ)
    off = np.concatenate(([0], np.cumsum(comp.trk_ncl.astype(np.int64))))
    steps = 0
    for t in range(comp.n_tracks):
        r0, n = off[t] - t, int(comp.trk_ncl[t]) - 1
        tr = compare_track(geo2, model, int(comp.trk_qpt[t]), int(comp.trk_sec0[t]), int(comp.trk_row0[t]), int(comp.trk_pad0[t]),
                           int(comp.trk_time0[t]), comp.a_rowdiff[r0:r0 + n], comp.a_secleg[r0:r0 + n], comp.a_padres[r0:r0 + n],
                           comp.a_timeres[r0:r0 + n], tag=f"c0 track {t}")
        steps += len(tr)
    assert steps == comp.n_attached - comp.n_tracks and steps > 10_000


# ---------------------------------------------------------------------------------------------- (b) crafted tracks
def test_consecutive_not_ok_steps(geo36):
    # |q/pT| = 127 and long outward row jumps: sp2 = sp + k*dx leaves [-0.95, 0.95] on several steps in a row (C3-6).
    # Reading 8: the prediction is then the PREVIOUS rebuilt cluster; C3-9: y,u re-seated on the cluster, sp = clamp(sp2),
    # dt unchanged.  Residuals are non-zero so that "previous cluster" differs from (0,0) and from the first cluster.
    model = Model(geo36, BZ)
    for qpt in (127, -127):
        tr = compare_track(geo36, model, qpt, 7, 5, 3000, 500_000,
                           rowdiff=[3, 60, 30, 25, 20, 1, 0, 5], secleg=[0, 0, 0, 0, 0, 0, 0x80, 0],
                           padres=[5, 700, 65000, 40, 9, 3, 2, 1], timeres=[100, -3000, 77, 12345, 5, 4, 3, 2], tag=f"notok qpt={qpt}")
        oks = [r["ok"] for r in tr]
        assert oks[0] == 1 and oks[1:5] == [0, 0, 0, 0], oks            # four consecutive impossible propagations
        for a, b in zip(tr[1:5], tr[0:4]):                               # reading 8: predicted = previous rebuilt cluster
            assert (a["P_pred"], a["T_pred"]) == (b["P"], b["T"])
        assert abs(f32(tr[2]["spn"])) == pytest.approx(0.95) and tr[2]["dtn"] == tr[1]["dtn"]   # sp clamped, dt untouched
        assert any(r["ok"] == 1 for r in tr[5:])                         # and the model recovers once the leg turns


def test_multi_step_rotations_both_ways(geo36):
    # C3-5: d = 2, 9 rotate by +2, +9 sector steps; d = 10, 16 by -8, -2 (d > n_az/2 goes the short way round); each
    # elementary rotation uses the OLD (x, y, sp).  A d that is rotated only once, or the wrong way, changes x/y/sp bits.
    model = Model(geo36, BZ)
    for d, want_sec in ((2, 6), (9, 13), (10, 14), (16, 2)):
        for qpt in (-30, 0, 45):
            tr = compare_track(geo36, model, qpt, 4, 40, 2900, 640_000, rowdiff=[1, 1, 2], secleg=[0, d, 0], padres=[3, 65530, 8],
                               timeres=[7, 65, -20], tag=f"rot d={d} qpt={qpt}")
            assert tr[1]["sec"] == want_sec
    # on side C the azimuth wraps inside the side (sector 18 + ...), several steps
    tr = compare_track(geo36, model, 20, 34, 100, 4000, 9000, rowdiff=[1, 1], secleg=[5, 0x80 | 14], padres=[0, 0], timeres=[0, 0], tag="rot side C")
    assert [r["sec"] for r in tr] == [18 + (16 + 5) % 18, 18 + (16 + 5 + 14) % 18]


def test_time_slope_saturates_and_time_prediction_clamps(geo36):
    model = Model(geo36, BZ)
    # huge time residuals drive dt to +DT_MAX, then to -DT_MAX (C3-9 clamp)
    tr = compare_track(geo36, model, 10, 3, 20, 3500, 100_000, rowdiff=[1] * 6, secleg=[0] * 6, padres=[0] * 6,
                       timeres=[900_000, 900_000, 5, -4_000_000, -4_000_000, 0], tag="dt saturation")
    dts = [f32(r["dtn"]) for r in tr]
    assert 8.0 in dts and -8.0 in dts
    # T0 just below 2^24 and a positive time slope: u2*64 passes 2^24 - 1 and T_pred clamps at 16777215 exactly (quantT)
    tr = compare_track(geo36, model, 0, 3, 20, 3500, 16_777_000, rowdiff=[1, 1, 1, 1], secleg=[0] * 4, padres=[0] * 4,
                       timeres=[150, 0, 0, 0], tag="T clamp")
    assert 16_777_215 in [r["T_pred"] for r in tr]
    # a first time code far above the format's range (adversarial): still one answer
    tr = compare_track(geo36, model, -5, 3, 20, 3500, 0xF000_0000, rowdiff=[1, 1], secleg=[0, 0], padres=[1, 2], timeres=[3, 4], tag="T huge")
    assert tr[0]["T_pred"] == 16_777_215


def test_pad_prediction_clamps_at_both_ends(geo36):
    model = Model(geo36, BZ)
    # P0 = 65535 is far outside the row (y large): the prediction on the next rows saturates at 65535
    tr = compare_track(geo36, model, 0, 2, 130, 65535, 50_000, rowdiff=[1, 1, 1], secleg=[0] * 3, padres=[0, 0, 0], timeres=[0] * 3, tag="P high")
    assert tr[0]["P_pred"] == 65535
    # P0 = 0 on the innermost rows and a sector step towards negative y: prediction clamps at 0
    tr = compare_track(geo36, model, 40, 2, 100, 0, 50_000, rowdiff=[20, 1], secleg=[1, 0], padres=[0, 0], timeres=[0] * 2, tag="P low")
    assert tr[0]["P_pred"] == 0


def test_start_direction_clamp(geo36):
    # C3-2: sd = clamp(0.5 k L): with |q/pT| = 127 and x > 160 cm the unclamped value exceeds 0.95 (sqrt of a negative
    # number without the clamp)
    model = Model(geo36, BZ)
    for qpt in (127, -127, -128):
        for row0 in (100, 140, 151):
            compare_track(geo36, model, qpt, 9, row0, 3200, 70_000, rowdiff=[0, 1], secleg=[0, 0x80], padres=[1, 2], timeres=[3, 4],
                          tag=f"init clamp qpt={qpt} row0={row0}")
    st = model.init(127, 140, 3200, 70_000)
    assert abs(float(st["sp"])) <= 0.95 and not np.isnan(st["sp"])


def test_out_of_format_bytes_are_reduced_first(geo36):
    # reading 19: rd = a_rowdiff mod n_rows (bytes 152..255), d = (a_secleg & 0x3F) mod n_az (18..63), bit 6 ignored --
    # on an inward leg too, where the row moves by n_rows - rd
    model = Model(geo36, BZ)
    tr = compare_track(geo36, model, -12, 20, 60, 3000, 300_000,
                       rowdiff=[200, 255, 152, 153, 3], secleg=[0x80, 0x40 | 35, 63, 0x80 | 18, 0xFF],
                       padres=[1, 2, 3, 4, 5], timeres=[10, 20, 30, 40, 50], tag="reading 19")
    rows, secs, dirs = [r["row"] for r in tr], [r["sec"] for r in tr], [r["dir"] for r in tr]
    assert dirs == [-1, -1, -1, +1, -1]
    assert rows == [(60 - 48) % 152, (12 - 103) % 152, 61, 62, (62 - 3) % 152]
    assert secs == [20, 18 + (2 + 17) % 18, 18 + (1 + 9) % 18, 28, 18 + (10 + 9) % 18]


# ---------------------------------------------------------------------------------------------- (c) random bytes
def test_random_byte_tracks(geo36):
    c = random_compressed(geo36, 1000, 0, seed=77, max_ncl=40)
    model = Model(geo36, BZ)
    off = np.concatenate(([0], np.cumsum(c.trk_ncl.astype(np.int64))))
    n_notok = n_multi = 0
    for t in range(c.n_tracks):
        r0, n = off[t] - t, int(c.trk_ncl[t]) - 1
        tr = compare_track(geo36, model, int(c.trk_qpt[t]), int(c.trk_sec0[t]), int(c.trk_row0[t]), int(c.trk_pad0[t]), int(c.trk_time0[t]),
                           c.a_rowdiff[r0:r0 + n], c.a_secleg[r0:r0 + n], c.a_padres[r0:r0 + n], c.a_timeres[r0:r0 + n], tag=f"random track {t}")
        n_notok += sum(1 for r in tr if not r["ok"])
        n_multi += int(np.count_nonzero(((c.a_secleg[r0:r0 + n] & 0x3F) % 18) > 1))
    assert n_notok > 1000 and n_multi > 10_000                       # the branches are exercised, not just present
