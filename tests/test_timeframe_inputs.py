"""The time-frame-scale torch generators (tmd_inputs/timeframe.py) produce valid, physical-looking workloads:
their truth survives the oracle codec byte for byte and has the shape BASELINE.json's configs describe."""
import numpy as np
import torch

from oracle import tmd_oracle as O
from tmd_inputs import build_geometry, physical as ph, timeframe as tf
from tmd_inputs.layout import CLUSTER_DTYPE, Compressed

BZ = 0.5


def truth_to_event(tr: tf.Truth) -> ph.Event:
    att = tr.att.cpu().numpy().view(CLUSTER_DTYPE).reshape(-1)
    return ph.Event(trk_ncl=tr.trk_ncl.cpu().numpy().view(np.uint16), trk_qptf=tr.trk_qptf.cpu().numpy(),
                    att=att, leg=tr.leg.cpu().numpy(), un=np.zeros(0, CLUSTER_DTYPE))


def test_truth_round_trips_through_the_oracle_codec():
    geo = build_geometry(36)
    for cfg in (ph.config2_like(1500, 0, seed=3), ph.config4_like(6000, 0, seed=5)):
        ev = truth_to_event(tf.generate_truth(cfg, geo, "cpu", batch=2000))
        assert len(ev.trk_ncl) == cfg.n_tracks and int(ev.trk_ncl.sum()) == len(ev.att)
        comp = O.encode(geo, BZ, ev.trk_ncl, ev.trk_qptf, ev.att, ev.leg, ev.un)
        cl, bo, _ = O.decode(geo, BZ, comp)
        want, want_bo = ph.canonical(ev, geo)
        assert np.array_equal(bo, want_bo) and cl.tobytes() == want.tobytes()
        # physical-looking: small residuals, rows advance by one almost always
        assert np.median(np.abs(comp.a_padres.astype(np.int16).astype(int))) <= 12
        assert np.median(np.abs(comp.a_timeres.astype(np.int32).astype(int))) <= 12
        assert (comp.a_rowdiff == 1).mean() > 0.97


def test_workload_shapes():
    geo = build_geometry(36)
    ev = truth_to_event(tf.generate_truth(ph.config2_like(4000, 0, seed=4), geo, "cpu"))
    ncl = ev.trk_ncl.astype(int)
    assert 105 < ncl.mean() < 140 and ncl.max() > 152 and ev.leg.max() >= 1       # ~120 clusters/track, 10 % loopers
    ev = truth_to_event(tf.generate_truth(ph.config4_like(20000, 0, seed=5), geo, "cpu"))
    ncl = ev.trk_ncl.astype(int)
    assert 25 < ncl.mean() < 50 and ncl.max() > 300 and ncl.min() == 1             # geometric(40) + long loopers


def test_unattached_truth_generator_through_the_oracle_codec():
    geo = build_geometry(36)
    un = tf.generate_unattached_truth(geo, 200_000, 3, "cpu").numpy().view(CLUSTER_DTYPE).reshape(-1)
    assert abs(len(un) - 200_000) < 5000
    c = O.encode(geo, BZ, np.zeros(0, np.uint16), np.zeros(0, np.float32), np.zeros(0, CLUSTER_DTYPE), np.zeros(0, np.uint8), un)
    c.check_shapes()
    assert int(c.u_bin_count.sum()) == c.n_unattached == len(un)
    cl, bo, _ = O.decode(geo, BZ, c)
    # density ~ 1/x(row); decoded times ascend inside a bin (sorted by the encoder); pads inside the row
    per_row = np.bincount(cl["row"], minlength=152)
    assert per_row[:10].mean() > 2.0 * per_row[-10:].mean()
    same = (cl["row"][1:] == cl["row"][:-1]) & (cl["sector"][1:] == cl["sector"][:-1])
    assert np.all(cl["time"][1:][same] >= cl["time"][:-1][same])
    assert cl["time"].max() < (1 << 24)
    assert np.all(cl["pad"] < geo.row_npads[cl["row"]].astype(np.int64) * 64)
