"""Cluster-domain event generator: exact helices in a uniform field + noise -> quantised TPC clusters.

Stand-in for the paper's real / Monte-Carlo time frames, which are not available;
recipe = SURVEY.md §8(d) and BASELINE.json `configs`.  The output is *cluster truth* (what an encoder would be
given): it contains NO arithmetic of the track-model codec.  Tests hand it to the oracle encoder to obtain a
compressed SoA, and compare decode(encode(x)) with `canonical(x)` built here with numpy library sorts.

All helix geometry is done in float64.  Frames: sector `az` has its local x axis at global angle (az+0.5)*20 deg,
local y counter-clockwise; sector = side*18 + az.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np

from .geometry import Geometry, TF_NBINS
from .layout import CLUSTER_DTYPE

KB_PER_TESLA = 0.00299792458      # curvature [1/cm] = KB_PER_TESLA * Bz[T] * q/pT[c/GeV]
DRIFT_CM_PER_BIN = 0.5
DRIFT_LEN_CM = 250.0
SECTOR_RAD = np.deg2rad(20.0)


@dataclass
class Event:
    """Cluster truth of one synthetic time frame."""
    trk_ncl: np.ndarray    # u16[n_tracks]
    trk_qptf: np.ndarray   # f32[n_tracks]  signed curvature / KB  (c/GeV), SURVEY C6
    att: np.ndarray        # CLUSTER_DTYPE[n_attached], g order (track after track)
    leg: np.ndarray        # u8[n_attached] leg index within the track
    un: np.ndarray         # CLUSTER_DTYPE[n_unattached], arbitrary order


@dataclass
class EventConfig:
    n_tracks: int
    n_unattached: int
    seed: int
    az_lo: int = 0                 # tracks are started inside sectors az_lo .. az_hi-1 (both sides unless one_side)
    az_hi: int = 18
    one_side: bool = False         # config 0: sectors 0,1 only (side A)
    confine: bool = False          # truncate a track when it leaves az_lo..az_hi-1 (config 0's wedge)
    pt_law: str = "power"          # "power": pdf ~ pT^-3 above pt_lo ; "loguniform": log-uniform pt_lo..pt_hi
    pt_lo: float = 0.15
    pt_hi: float = 10.0
    eta_max: float = 0.9
    looper_frac: float = 0.0       # fraction of tracks drawn with pT in looper_pt and up to looper_legs legs
    looper_pt: tuple = (0.10, 0.18)
    looper_legs: int = 3
    looper_eta_max: float = 0.9    # loopers with small |eta| stay inside the drift volume for more legs
    full_len_frac: float = 0.6     # fraction of tracks allowed the full 152 clusters; the rest capped U(len_lo,len_hi)
    len_lo: int = 20
    len_hi: int = 152
    len_law: str = "cap"           # "cap" as above, "geometric": cap ~ Geometric(mean len_mean) clipped to [1,152]
    len_mean: float = 40.0
    min_ncl: int = 20              # tracks with fewer clusters are dropped (and replaced)
    row0_max: int = 0              # first row drawn uniformly in 0..row0_max (secondaries start late)
    unatt_law: str = "uniform"     # "uniform" over bins or "inv_x" (density ~ 1/x(row))
    single_event: bool = True      # one common t0 (else t0 uniform over the time frame)
    noise_cm: float = 0.05
    bz_tesla: float = 0.5


def _copy_through(rng: np.random.Generator, n: int):
    """qTot/qMax/sigmas/flags (BASELINE.json config 0 recipe; Moyal stand-in for Landau)."""
    z = rng.standard_normal(n)
    moyal = -np.log(np.maximum(z * z, 1e-300))
    qtot = np.clip(np.rint(60.0 + 15.0 * moyal), 1, 65535)
    qmax = np.clip(np.rint(qtot * rng.uniform(0.2, 0.6, n)), 1, qtot)
    sigpad = np.clip(np.rint(rng.normal(40.0, 10.0, n)), 0, 255)
    sigtime = np.clip(np.rint(rng.normal(40.0, 10.0, n)), 0, 255)
    flags = rng.integers(0, 256, n)
    return qtot.astype(np.uint16), qmax.astype(np.uint16), sigpad.astype(np.uint8), sigtime.astype(np.uint8), flags.astype(np.uint8)


def _draw_tracks(cfg: EventConfig, rng: np.random.Generator, n: int):
    u = rng.random(n)
    if cfg.pt_law == "power":
        pt = np.minimum(cfg.pt_lo * (1.0 - u) ** -0.5, 50.0)
    else:
        pt = np.exp(np.log(cfg.pt_lo) + u * (np.log(cfg.pt_hi) - np.log(cfg.pt_lo)))
    looper = rng.random(n) < cfg.looper_frac
    pt = np.where(looper, rng.uniform(cfg.looper_pt[0], cfg.looper_pt[1], n), pt)
    max_legs = np.where(looper, rng.integers(2, cfg.looper_legs + 1, n) if cfg.looper_legs >= 2 else 1, 1)
    charge = np.where(rng.random(n) < 0.5, -1.0, 1.0)
    eta = rng.uniform(-cfg.eta_max, cfg.eta_max, n)
    eta = np.where(looper, eta * (cfg.looper_eta_max / cfg.eta_max), eta)
    if cfg.one_side:
        eta = np.abs(eta)
    span = (cfg.az_hi - cfg.az_lo) * SECTOR_RAD
    phi0 = cfg.az_lo * SECTOR_RAD + rng.random(n) * span
    if cfg.len_law == "geometric":
        cap = np.clip(rng.geometric(1.0 / cfg.len_mean, n), 1, 152)
    else:
        cap = np.where(rng.random(n) < cfg.full_len_frac, 152, rng.integers(cfg.len_lo, cfg.len_hi + 1, n))
    cap = np.where(looper, 152 * max_legs, cap)
    row0 = rng.integers(0, cfg.row0_max + 1, n)
    t0 = np.full(n, 2000.0) if cfg.single_event else rng.uniform(0.0, TF_NBINS - 500.0, n)
    z0 = rng.normal(0.0, 5.0, n)
    return pt, charge, eta, phi0, cap.astype(np.int64), row0.astype(np.int64), max_legs.astype(np.int64), t0, z0


def _trace(cfg: EventConfig, geo: Geometry, rng: np.random.Generator, n: int):
    """Follow n helices row by row.  Returns per-cluster arrays (track id, leg, sector, row, P, T) in walk order."""
    pt, charge, eta, phi0, cap, row0, max_legs, t0, z0 = _draw_tracks(cfg, rng, n)
    kappa = charge * KB_PER_TESLA * cfg.bz_tesla / pt          # signed curvature d(phi)/ds, 1/cm
    circ = 2.0 * np.pi / np.abs(kappa)
    tanl = np.sinh(eta)
    side = (eta < 0).astype(np.int64)
    az = np.floor(phi0 / SECTOR_RAD).astype(np.int64) % 18
    az0 = az.copy()
    row_cur = row0 - 1
    dirn = np.ones(n, np.int64)
    leg = np.zeros(n, np.int64)
    s_prev = np.zeros(n)
    alive = np.ones(n, bool)
    ncl = np.zeros(n, np.int64)
    miss = np.zeros(n, np.int64)
    last_hit = row0.copy()
    half_w = (geo.row_npads.astype(np.float64) / 2.0) * geo.row_padw_f64      # half width of the pad row, cm
    out = []
    S_MAX = 0.9
    offsets = np.array([0, 1, -1, 2, -2])
    for _ in range(152 * 6 + 128):
        idx = np.nonzero(alive)[0]
        if idx.size == 0:
            break
        cand = row_cur[idx] + dirn[idx]
        # leaving the row range: outward -> exits the TPC; inward -> passes the inner field cage, next leg outward
        ex_out = cand > 151
        ex_in = cand < 0
        more = leg[idx] + 1 < max_legs[idx]
        kill = ex_out | (ex_in & ~more)
        alive[idx[kill]] = False
        flip = ex_in & more
        fi = idx[flip]
        leg[fi] += 1; dirn[fi] = 1; row_cur[fi] = -1; miss[fi] = 0
        az[fi] = az0[fi]                      # a circle through the beam line comes out again where it first did
        keep = ~(kill | flip)
        idx = idx[keep]; cand = cand[keep]
        if idx.size == 0:
            continue
        xr = geo.row_x_f64[cand]
        k = kappa[idx]
        best_s = np.full(idx.size, np.inf); best_y = np.zeros(idx.size); best_az = np.zeros(idx.size, np.int64)
        for o in offsets:
            a = (az[idx] + o) % 18
            alpha = (a + 0.5) * SECTOR_RAD
            p0 = phi0[idx] - alpha
            S = np.sin(p0) + k * xr
            okS = np.abs(S) <= S_MAX
            Sc = np.clip(S, -1.0, 1.0)
            pl = np.where(dirn[idx] > 0, np.arcsin(Sc), np.pi - np.arcsin(Sc))
            s = np.mod((pl - p0) / k, circ[idx])
            s = s + np.ceil(np.maximum(s_prev[idx] - s, 0.0) / circ[idx]) * circ[idx]
            s = np.where(s <= s_prev[idx], s + circ[idx], s)
            y = (np.cos(p0) - np.cos(pl)) / k
            good = okS & (np.abs(y) < half_w[cand]) & (s - s_prev[idx] < 0.6 * circ[idx]) & (s < best_s)
            if cfg.confine:
                good &= (a >= cfg.az_lo) & (a < cfg.az_hi)
            best_s = np.where(good, s, best_s); best_y = np.where(good, y, best_y); best_az = np.where(good, a, best_az)
        found = np.isfinite(best_s)
        z = z0[idx] + best_s * tanl[idx]
        found &= np.abs(z) < DRIFT_LEN_CM
        # misses: skip the row; too many misses -> turn inward (outward leg of a looper) or stop
        mi = idx[~found]
        miss[mi] += 1
        row_cur[mi] = cand[~found]
        too = miss[mi] > 6
        turn = too & (dirn[mi] > 0) & (leg[mi] + 1 < max_legs[mi])
        ti = mi[turn]
        leg[ti] += 1; dirn[ti] = -1; miss[ti] = 0; row_cur[ti] = last_hit[ti] + 1   # re-cross the last row on the way back
        alive[mi[too & ~turn]] = False
        # hits
        hi = idx[found]
        if hi.size:
            r = cand[found]
            y = best_y[found] + rng.normal(0.0, cfg.noise_cm, hi.size)
            zz = z[found] + rng.normal(0.0, cfg.noise_cm, hi.size)
            u = t0[hi] + (DRIFT_LEN_CM - np.abs(zz)) / DRIFT_CM_PER_BIN
            npads = geo.row_npads[r].astype(np.float64)
            P = np.clip(np.rint((y / geo.row_padw_f64[r] + npads / 2.0) * 64.0), 0, npads * 64 - 1).astype(np.int64)
            T = np.clip(np.rint(u * 64.0), 0, (1 << 24) - 1).astype(np.int64)
            out.append((hi, leg[hi].copy(), side[hi] * 18 + best_az[found], r, P, T))
            az[hi] = best_az[found]; row_cur[hi] = r; last_hit[hi] = r; s_prev[hi] = best_s[found]; miss[hi] = 0
            ncl[hi] += 1
            alive[hi[ncl[hi] >= cap[hi]]] = False
    if not out:
        z = np.zeros(0, np.int64)
        return (z,) * 6, ncl, (kappa / (KB_PER_TESLA * cfg.bz_tesla))
    cols = [np.concatenate(c) for c in zip(*out)]
    order = np.argsort(cols[0], kind="stable")      # group by track, keep walk order inside the track
    return tuple(c[order] for c in cols), ncl, (kappa / (KB_PER_TESLA * cfg.bz_tesla))


def generate_event(cfg: EventConfig, geo: Geometry) -> Event:
    rng = np.random.Generator(np.random.Philox(key=cfg.seed))
    n_draw = int(cfg.n_tracks * 1.6) + 64
    (tid, leg, sec, row, P, T), ncl, qpt = _trace(cfg, geo, rng, n_draw)
    good = np.nonzero(ncl >= cfg.min_ncl)[0][: cfg.n_tracks]
    if good.size < cfg.n_tracks:
        raise RuntimeError(f"only {good.size} of {cfg.n_tracks} tracks survived; raise the oversampling")
    sel = np.zeros(n_draw, bool); sel[good] = True
    m = sel[tid]
    tid, leg, sec, row, P, T = (c[m] for c in (tid, leg, sec, row, P, T))
    n_att = tid.size
    att = np.zeros(n_att, CLUSTER_DTYPE)
    att["sector"], att["row"], att["pad"], att["time"] = sec, row, P, T
    att["qtot"], att["qmax"], att["sigpad"], att["sigtime"], att["flags"] = _copy_through(rng, n_att)
    # unattached
    n_un = cfg.n_unattached
    n_bins = geo.n_bins
    w = np.ones(n_bins) if cfg.unatt_law == "uniform" else np.tile(1.0 / geo.row_x_f64, geo.n_sectors_out)
    b = rng.choice(n_bins, size=n_un, p=w / w.sum())
    un = np.zeros(n_un, CLUSTER_DTYPE)
    un["sector"], un["row"] = b // geo.n_rows, b % geo.n_rows
    un["pad"] = (rng.random(n_un) * geo.row_npads[b % geo.n_rows] * 64).astype(np.uint16)
    if cfg.single_event:
        un["time"] = ((2000.0 + rng.random(n_un) * 500.0) * 64).astype(np.uint32)
    else:
        un["time"] = (rng.random(n_un) * TF_NBINS * 64).astype(np.uint32)
    un["qtot"], un["qmax"], un["sigpad"], un["sigtime"], un["flags"] = _copy_through(rng, n_un)
    return Event(trk_ncl=ncl[good].astype(np.uint16), trk_qptf=qpt[good].astype(np.float32),
                 att=att, leg=leg.astype(np.uint8), un=un)


def canonical(ev: Event, geo: Geometry):
    """The decoder's expected output for cluster truth `ev`, built with numpy library sorts only:
    per bin, attached clusters in ascending g (stable argsort by bin), then unattached clusters ascending by
    (time,pad,qtot,qmax,sigpad,sigtime,flags) (lexsort).  Returns (clusters, bin_offset)."""
    n_bins = geo.n_bins
    ab = ev.att["sector"].astype(np.int64) * geo.n_rows + ev.att["row"]
    ub = ev.un["sector"].astype(np.int64) * geo.n_rows + ev.un["row"]
    a_sorted = ev.att[np.argsort(ab, kind="stable")]
    u_order = np.lexsort((ev.un["flags"], ev.un["sigtime"], ev.un["sigpad"], ev.un["qmax"], ev.un["qtot"],
                          ev.un["pad"], ev.un["time"], ub))
    u_sorted = ev.un[u_order]
    a_cnt = np.bincount(ab, minlength=n_bins); u_cnt = np.bincount(ub, minlength=n_bins)
    bin_offset = np.zeros(n_bins + 1, np.uint32)
    bin_offset[1:] = np.cumsum(a_cnt + u_cnt)
    out = np.zeros(len(ev.att) + len(ev.un), CLUSTER_DTYPE)
    a_start = np.concatenate(([0], np.cumsum(a_cnt)))[:-1]
    u_start = np.concatenate(([0], np.cumsum(u_cnt)))[:-1]
    a_dst = bin_offset[:-1].astype(np.int64)[np.sort(ab, kind="stable")] + (np.arange(len(ab)) - a_start[np.sort(ab, kind="stable")])
    u_dst = (bin_offset[:-1].astype(np.int64) + a_cnt)[ub[u_order]] + (np.arange(len(ub)) - u_start[ub[u_order]])
    out[a_dst] = a_sorted
    out[u_dst] = u_sorted
    return out, bin_offset


# --- BASELINE.json configs in the cluster domain (c0, c1 at full size; c2-c4 mixes at reduced size for tests) -------

def config0() -> EventConfig:
    """tiny: 2 sectors, 200 tracks log-uniform pT 0.1-10 GeV, 20-152 clusters, 5000 unattached, seed 1."""
    return EventConfig(n_tracks=200, n_unattached=5000, seed=1, az_lo=0, az_hi=2, one_side=True, confine=True,
                       pt_law="loguniform", pt_lo=0.1, pt_hi=10.0, full_len_frac=0.0, len_lo=20, len_hi=152,
                       min_ncl=20, unatt_law="uniform", single_event=True)


def config1(n_tracks: int = 10_000, n_unattached: int = 300_000, seed: int = 2) -> EventConfig:
    """single central Pb-Pb-like event: power-law pT, 10% multi-leg loopers, 1/x unattached density."""
    return EventConfig(n_tracks=n_tracks, n_unattached=n_unattached, seed=seed, pt_law="power", pt_lo=0.15,
                       looper_frac=0.10, full_len_frac=0.75, len_lo=20, len_hi=152, min_ncl=20, row0_max=0,
                       unatt_law="inv_x", single_event=True)


def config2_like(n_tracks: int, n_unattached: int, seed: int = 3) -> EventConfig:
    """time-frame mix (c2/c3 shape): as config 1 but t0 spread over the time frame."""
    c = config1(n_tracks, n_unattached, seed)
    c.single_event = False
    return c


def config4_like(n_tracks: int, n_unattached: int, seed: int = 5) -> EventConfig:
    """pp-like skew: geometric(40) lengths + 2% long multi-leg loopers."""
    return EventConfig(n_tracks=n_tracks, n_unattached=n_unattached, seed=seed, pt_law="power", pt_lo=0.15,
                       looper_frac=0.02, looper_legs=5, looper_eta_max=0.2, len_law="geometric", len_mean=40.0, min_ncl=1, row0_max=100,
                       unatt_law="inv_x", single_event=False)
