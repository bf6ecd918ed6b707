"""Pins for the four oracle lines that survived the round-2 mutation run (What's weak #1).  All CPU-only.

  (a) trk_qpt quantisation: trk_qpt = clamp(floor(16 * qpt + 0.5), -127, 127) -- expected values worked
      out by hand below, not computed with the formula;
  (b) the unattached sort key, C6 / C7-10 ("unassigned clusters are sorted by coordinate position ... stored as
      differences relative to the preceding cluster"): (time, pad, qtot, qmax, sigpad, sigtime, flags) in THAT order -- a
      hand-ordered bin in which every adjacent pair of key fields decides one comparison, and a 10 000-cluster heavy-tie bin
      against numpy.lexsort (a library sort, not the oracle's comparator);
  (c) C3-9's else branch (abs(s) < S_MIN => sp = clamp(sp2), dt unchanged) on steps with dx != 0: only a sector rotation
      can leave the track a hair's breadth from the next row's x; such steps are constructed below and every trace column
      is compared with the independent numpy-float32 evaluation tests/c3_numpy.py;
  (d) the oracle compiled with -fsanitize=address,undefined runs config 0 and 1000 random-byte tracks clean.

The oracle's arithmetic is not touched by this file's commit.
"""
import os
import subprocess
import sys

import numpy as np
import pytest

from c3_numpy import Model
from oracle import tmd_oracle as O
from test_oracle_independent import compare_track, f32
from tmd_inputs.layout import CLUSTER_DTYPE

BZ = 0.5
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


# ------------------------------------------------------------------------------------------------------- (a) trk_qpt
def test_trk_qpt_rounds_half_up_and_clamps_at_127(geo36):
    # 16*q + 0.5, then floor, then clamp to [-127, 127]; every product and sum below is exact in binary32
    cases = [
        (0.03125, 1),      # 0.5 + 0.5 = 1.0 -> 1            (plain floor(16 q) would give 0)
        (-0.03125, 0),     # -0.5 + 0.5 = 0.0 -> 0           (round-half-away would give -1)
        (0.09375, 2),      # 1.5 + 0.5 = 2.0 -> 2
        (-0.09375, -1),    # -1.5 + 0.5 = -1.0 -> -1         (round-half-even / half-away would give -2)
        (0.15625, 3),      # 2.5 + 0.5 = 3.0 -> 3            (round-half-even would give 2)
        (0.2, 3),          # 3.2 + 0.5 = 3.7 -> 3
        (-0.2, -3),        # -3.2 + 0.5 = -2.7 -> -3         (truncation would give -2)
        (7.90625, 127),    # 126.5 + 0.5 = 127.0 -> 127      (a clamp at 126 would give 126)
        (-7.90625, -126),  # -126.5 + 0.5 = -126.0 -> -126
        (7.96875, 127),    # 127.5 + 0.5 = 128.0 -> 128 -> clamp 127
        (-7.96875, -127),  # -127.5 + 0.5 = -127.0 -> -127   (a clamp at -126 would give -126)
        (8.0, 127),        # 128.5 -> 128 -> 127
        (-8.0, -127),      # -128 + 0.5 = -127.5 -> floor -128 -> clamp -127  (int8 -128 must never be stored)
        (100.0, 127), (-100.0, -127), (0.0, 0),
    ]
    n = len(cases)
    att = np.zeros(n, CLUSTER_DTYPE)
    att["row"] = 10; att["sector"] = 3; att["pad"] = 2000; att["time"] = 5000
    comp = O.encode(geo36, BZ, np.ones(n, np.uint16), np.array([q for q, _ in cases], np.float32), att, np.zeros(n, np.uint8),
                    np.zeros(0, CLUSTER_DTYPE))
    assert comp.trk_qpt.tolist() == [w for _, w in cases]


# ------------------------------------------------------------------------------------------------------- (b) sort key
def _decoded_fields(comp, lo, hi):
    """(time, pad, qtot, qmax, sigpad, sigtime, flags) rows of the unattached clusters [lo, hi) of ONE bin, in stored order."""
    time = np.cumsum(comp.u_timediff[lo:hi].astype(np.uint64)) & 0xFFFFFFFF
    pad = np.cumsum(comp.u_paddiff[lo:hi].astype(np.uint64)) & 0xFFFF
    return list(zip(time.tolist(), pad.tolist(), comp.u_qtot[lo:hi].tolist(), comp.u_qmax[lo:hi].tolist(), comp.u_sigpad[lo:hi].tolist(),
                    comp.u_sigtime[lo:hi].tolist(), comp.u_flags[lo:hi].tolist()))


def _unattached(rows, sector, row):
    un = np.zeros(len(rows), CLUSTER_DTYPE)
    for i, (t, p, qt, qm, sp, st, fl) in enumerate(rows):
        un[i] = (t, p, qt, qm, sp, st, fl, row, sector, 0)
    return un


def test_unattached_sort_key_order_by_hand(geo36):
    assert CLUSTER_DTYPE.names == ("time", "pad", "qtot", "qmax", "sigpad", "sigtime", "flags", "row", "sector", "zero")
    # (time, pad, qtot, qmax, sigpad, sigtime, flags).  Listed in the order the encoder must emit them; each neighbour pair is
    # decided by ONE field while every later field pulls the other way, so swapping any two adjacent key fields reorders it.
    want = [
        (999, 65535, 9, 9, 9, 9, 9),            # time decides (pad, and all the rest, larger)
        (1000, 639, 65535, 9, 9, 9, 9),         # pad decides against the next (qtot larger)
        (1000, 640, 4, 60000, 255, 255, 255),   # qtot decides (qmax .. flags larger)
        (1000, 640, 5, 8, 200, 200, 200),       # qmax decides (sigpad .. larger)
        (1000, 640, 5, 9, 2, 9, 9),             # sigpad decides (sigtime, flags larger)
        (1000, 640, 5, 9, 3, 2, 7),             # sigtime decides (flags larger)
        (1000, 640, 5, 9, 3, 3, 0),             # flags decides
        (1000, 640, 5, 9, 3, 3, 1),
        (1000, 640, 5, 9, 3, 3, 1),             # an exact duplicate stays (both emitted)
        (1000, 640, 6, 0, 0, 0, 0),
        (1001, 0, 0, 0, 0, 0, 0),
    ]
    shuffled = [want[i] for i in (7, 9, 10, 5, 0, 3, 8, 6, 1, 4, 2)]
    comp = O.encode(geo36, BZ, np.zeros(0, np.uint16), np.zeros(0, np.float32), np.zeros(0, CLUSTER_DTYPE), np.zeros(0, np.uint8),
                    _unattached(shuffled, sector=5, row=77))
    b = 5 * geo36.n_rows + 77
    assert comp.u_bin_count[b] == len(want) and comp.u_bin_count.sum() == len(want)
    assert _decoded_fields(comp, 0, len(want)) == want
    # first of the bin: difference to (0, 0); then to the predecessor, mod 2^16 / 2^32
    assert comp.u_timediff[:3].tolist() == [999, 1, 0] and comp.u_paddiff[:3].tolist() == [65535, (639 - 65535) % 65536, 1]


def test_unattached_sort_key_heavy_ties_against_lexsort(geo36):
    rng = np.random.default_rng(515)
    n = 10_000
    # few distinct values per field: (time, pad) ties are the rule, and every later field gets to decide many comparisons
    f = {"time": rng.integers(100, 104, n), "pad": rng.integers(64, 67, n) * 64, "qtot": rng.integers(10, 13, n), "qmax": rng.integers(0, 3, n),
         "sigpad": rng.integers(5, 8, n), "sigtime": rng.integers(250, 253, n), "flags": rng.integers(0, 3, n)}
    un = np.zeros(n, CLUSTER_DTYPE)
    for k, v in f.items():
        un[k] = v
    un["sector"] = 35; un["row"] = 151
    comp = O.encode(geo36, BZ, np.zeros(0, np.uint16), np.zeros(0, np.float32), np.zeros(0, CLUSTER_DTYPE), np.zeros(0, np.uint8), un)
    order = np.lexsort((f["flags"], f["sigtime"], f["sigpad"], f["qmax"], f["qtot"], f["pad"], f["time"]))   # last key = primary
    want = list(zip(*(f[k][order].tolist() for k in ("time", "pad", "qtot", "qmax", "sigpad", "sigtime", "flags"))))
    assert comp.u_bin_count[geo36.n_bins - 1] == n
    assert _decoded_fields(comp, 0, n) == want


# ------------------------------------------------------------------------------------------- (c) abs(s) < S_MIN with dx != 0
def _short_steps_after_a_rotation(geo, model, want: int):
    """Tracks whose FIRST step rotates by one sector and lands within ~0.5 um .. 9 um of the target row's x: the start pad is
    solved from x' = x cos(a) +- y sin(a) = row_x[target], then the step is evaluated with tests/c3_numpy.py and kept only if
    it really has ok = 1, dx != 0 and abs(s) < S_MIN."""
    row_x, padw, npads = np.asarray(geo.row_x, np.float64), np.asarray(geo.row_padw, np.float64), np.asarray(geo.row_npads)
    ca, sa = float(geo.cos_a), float(geo.sin_a)
    found = []
    rng = np.random.default_rng(909)
    while len(found) < want:
        row0 = int(rng.integers(20, geo.n_rows))
        d = int(rng.choice([1, geo.n_az - 1]))                      # one sector up / one sector down
        sn = sa if d == 1 else -sa
        target = int(rng.integers(0, geo.n_rows))
        y = (row_x[target] - row_x[row0] * ca) / sn                 # x' = x ca + y sn
        pad = y / padw[row0] + npads[row0] // 2
        if not (1.0 < pad < npads[row0] - 1.0):
            continue
        qpt = int(rng.choice([-127, -90, -40, 40, 90, 127]))
        for P0 in (int(round(pad * 64)) + k for k in (-1, 0, 1)):
            rd = (target - row0) % geo.n_rows
            st = model.init(qpt, row0, P0, 6400)
            with np.errstate(all="ignore"):
                tr, *_ = model.step(dict(st), 4, row0, P0, 6400, 1, rd, d, 0, 0)
            if not tr["ok"] or tr["s"] is None:
                continue
            dx = np.float32(model.row_x[target]) - np.float32(f32(tr["x"]))
            if dx != 0 and abs(f32(tr["s"])) < 0.001:
                found.append((qpt, row0, P0, rd, d, float(dx), f32(tr["s"])))
                break
    return found


def test_short_step_with_nonzero_dx_takes_sp2(geo36):
    model = Model(geo36, BZ)
    cases = _short_steps_after_a_rotation(geo36, model, 40)
    assert len(cases) >= 20
    n_sp_moves = 0
    for i, (qpt, row0, P0, rd, d, dx, s) in enumerate(cases):
        assert dx != 0 and abs(s) < 0.001
        # the short step, then three ordinary ones that carry its sp and dt forward (a wrong sp shifts their predictions)
        tr = compare_track(geo36, model, qpt, 4, row0, P0, 6400, rowdiff=[rd, 1, 1, 2], secleg=[d, 0, 0, 0], padres=[3, -2, 1, 0],
                           timeres=[5, -4, 2, 1], tag=f"short step {i}")
        first = tr[0]
        assert first["ok"] == 1 and abs(f32(first["s"])) < 0.001
        assert first["spn"] == first["sp2"] or abs(f32(first["sp2"])) > 0.95        # sp <- clamp(sp2): the else branch of C3-9
        assert first["dtn"] == 0                                                    # dt untouched (still the initial +0.0)
        n_sp_moves += first["sp2"] != first["sp"]
    assert n_sp_moves >= 20, "the pin needs steps where clamp(sp2) differs from the old sp"


# ------------------------------------------------------------------------------------------------------- (d) sanitizers
def test_oracle_under_address_and_undefined_behaviour_sanitizers(tmp_path):
    """the oracle under ASan + UBSan.  The sanitised library is built next to the test's temp files and driven by a
    child interpreter with libasan preloaded; it encodes + decodes config 0 and decodes 1000 random-byte tracks plus
    unattached clusters.  Any report makes the child exit non-zero (halt_on_error, -fno-sanitize-recover)."""
    from oracle import build as OB
    libasan = subprocess.run(["gcc", "-print-file-name=libasan.so"], capture_output=True, text=True).stdout.strip()
    if not os.path.isabs(libasan) or not os.path.exists(libasan):
        pytest.skip("gcc has no libasan on this machine")
    san = str(tmp_path / "liborc_san.so")
    flags = [f for f in OB.CFLAGS if f != "-O2"] + ["-O1", "-g", "-fsanitize=address,undefined", "-fno-sanitize-recover=all", "-fno-omit-frame-pointer"]
    subprocess.run(["gcc", *flags, "-o", san, *OB.SRCS, "-lm"], check=True)
    child = f"""
import sys
sys.path.insert(0, {ROOT!r})
import numpy as np
from oracle import build as OB
OB.build = lambda force=False: {san!r}                      # the front end loads the sanitised library
from oracle import tmd_oracle as O
from tmd_inputs import build_geometry, physical as ph
from tmd_inputs.adversarial import random_compressed
geo = build_geometry(2)
ev = ph.generate_event(ph.config0(), geo)
comp = O.encode(geo, 0.5, ev.trk_ncl, ev.trk_qptf, ev.att, ev.leg, ev.un)
cl, bo, pr = O.decode(geo, 0.5, comp, probe_step=0xFFFFFFFF)
assert len(cl) == comp.n_attached + comp.n_unattached
geo36 = build_geometry(36)
c = random_compressed(geo36, 1000, 20000, 4242, max_ncl=60)
cl, bo, pr = O.decode(geo36, 0.5, c, probe_step=3)
assert int(bo[-1]) <= len(cl)
print("sanitised oracle ok", len(cl))
"""
    env = dict(os.environ, LD_PRELOAD=libasan, ASAN_OPTIONS="detect_leaks=0:halt_on_error=1:abort_on_error=0",
               UBSAN_OPTIONS="halt_on_error=1:print_stacktrace=1")
    r = subprocess.run([sys.executable, "-c", child], capture_output=True, text=True, env=env, timeout=600)
    assert r.returncode == 0 and "sanitised oracle ok" in r.stdout, r.stdout[-2000:] + r.stderr[-4000:]
    assert "runtime error" not in r.stderr and "AddressSanitizer" not in r.stderr, r.stderr[-4000:]
