import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def geo36():
    from tmd_inputs import build_geometry
    return build_geometry(36)


@pytest.fixture(scope="session")
def geo2():
    from tmd_inputs import build_geometry
    return build_geometry(2)


def parse_golden_trace(path):
    """tests/golden/c9_trace.txt -> dict(track, res, init, steps, out)."""
    out = {"res": [], "steps": [], "out": []}
    for line in open(path):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        k, *v = line.split()
        iv = [int(x, 0) for x in v]
        if k == "track":
            out["track"] = iv
        elif k == "res":
            out["res"].append(iv)
        elif k == "init":
            out["init"] = iv
        elif k == "step":
            out["steps"].append(iv)
        elif k == "out":
            out["out"].append(iv)
    return out


def residual_meta(ev):
    """Per residual entry (attached clusters with j>=1): track id, j, leg, clusters since the leg started."""
    ncl = ev.trk_ncl.astype(np.int64)
    off = np.concatenate(([0], np.cumsum(ncl)))
    t_of = np.repeat(np.arange(len(ncl)), ncl)
    j = np.arange(len(ev.att)) - off[t_of]
    chg = np.ones(len(ev.att), bool)
    chg[1:] = (ev.leg[1:] != ev.leg[:-1]) | (t_of[1:] != t_of[:-1])
    idx = np.arange(len(ev.att))
    since = idx - np.maximum.accumulate(np.where(chg, idx, 0))
    m = j >= 1
    return t_of[m], j[m], ev.leg[m].astype(np.int64), since[m]
