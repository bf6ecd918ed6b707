"""Time-frame-scale synthetic inputs on a torch device (what bench.py decodes; stand-ins for the paper's real / MC time
frames; recipe = SURVEY.md §8(d), BASELINE.json `configs`).

Two generators, neither containing arithmetic of the track-model codec:

* `generate_truth`  -- the same helix event model as `physical.py` (exact circles through the beam line in a uniform
  field, row crossings per sector frame, sector changes, looper legs, Gaussian noise, drift time), written with torch
  ops so that 2-3 M tracks / 240 M clusters are generated on the GPU in seconds.  Output = cluster truth of the
  ATTACHED clusters (g-ordered 16-byte records + leg index + per-track length and curvature).  It becomes the compressed
  SoA through an encoder: the oracle's in tests, the library's `tmd_encode_attached` in bench.py.
* `generate_unattached_truth` -- the UNATTACHED clusters in the cluster domain (per-bin counts Poisson around a 1/x(row)
  density, pad uniform over the row, time uniform over the frame, arbitrary order inside a bin): truth for an encoder.

Random numbers come from a seeded torch.Generator on the target device (CPU and CUDA streams differ; a run is
reproducible per device).
"""
from __future__ import annotations

import math
from dataclasses import dataclass

import numpy as np
import torch

from .geometry import Geometry, TF_NBINS
from .physical import DRIFT_CM_PER_BIN, DRIFT_LEN_CM, KB_PER_TESLA, EventConfig, config1, config2_like, config4_like

SECTOR_RAD = math.radians(20.0)


@dataclass
class Truth:
    """Attached-cluster truth on a torch device."""
    trk_ncl: torch.Tensor    # int16 (bits of u16) [n_tracks]
    trk_qptf: torch.Tensor   # float32 [n_tracks]
    att: torch.Tensor        # int32 [n_attached, 4] = 16-byte cluster records (layout.CLUSTER_DTYPE)
    leg: torch.Tensor        # uint8 [n_attached]
    un: torch.Tensor | None = None   # int32 [n_unattached, 4] unattached clusters, any order (set by whoever draws them)

    @property
    def n_tracks(self) -> int:
        return int(self.trk_ncl.shape[0])

    @property
    def n_attached(self) -> int:
        return int(self.leg.shape[0])


def _copy_through(gen, n, device):
    """qTot/qMax/sigmas/flags: Moyal stand-in for Landau(mpv 60, width 15), N(40,10) sigmas, uniform flags."""
    z = torch.randn(n, generator=gen, device=device, dtype=torch.float32)
    moyal = -torch.log(torch.clamp_min(z * z, 1e-30))
    qtot = torch.clamp(torch.round(60.0 + 15.0 * moyal), 1, 65535)
    qmax = torch.clamp(torch.round(qtot * (0.2 + 0.4 * torch.rand(n, generator=gen, device=device))), min=1.0)
    qmax = torch.minimum(qmax, qtot)
    sigpad = torch.clamp(torch.round(40.0 + 10.0 * torch.randn(n, generator=gen, device=device)), 0, 255)
    sigtime = torch.clamp(torch.round(40.0 + 10.0 * torch.randn(n, generator=gen, device=device)), 0, 255)
    flags = torch.randint(0, 256, (n,), generator=gen, device=device)
    return qtot.to(torch.int64), qmax.to(torch.int64), sigpad.to(torch.int64), sigtime.to(torch.int64), flags


def pack_records(time, pad, qtot, qmax, sigpad, sigtime, flags, row, sector) -> torch.Tensor:
    """int64 field tensors -> int32 [n,4] little-endian 16-byte records (layout only)."""
    w0 = time
    w1 = pad | (qtot << 16)
    w2 = qmax | (sigpad << 16) | (sigtime << 24)
    w3 = flags | (row << 8) | (sector << 16)
    return torch.stack([w0, w1, w2, w3], dim=1).to(torch.int32)   # int64 -> int32 conversion wraps (keeps the low 32 bits)


def _trace(cfg: EventConfig, geo: Geometry, gen, n: int, device):
    """Follow n helices row by row (vectorised over tracks).  Returns hit columns in walk order + per-track ncl, q/pT."""
    f64 = dict(device=device, dtype=torch.float64)
    rnd = lambda: torch.rand(n, generator=gen, **f64)
    row_x = torch.as_tensor(geo.row_x_f64, **f64)
    padw = torch.as_tensor(geo.row_padw_f64, **f64)
    npads = torch.as_tensor(geo.row_npads.astype(np.float64), **f64)
    half_w = npads / 2.0 * padw
    # --- track parameters
    u = rnd()
    if cfg.pt_law == "power":
        pt = torch.clamp_max(cfg.pt_lo * (1.0 - u) ** -0.5, 50.0)
    else:
        pt = torch.exp(math.log(cfg.pt_lo) + u * (math.log(cfg.pt_hi) - math.log(cfg.pt_lo)))
    looper = rnd() < cfg.looper_frac
    pt = torch.where(looper, cfg.looper_pt[0] + rnd() * (cfg.looper_pt[1] - cfg.looper_pt[0]), pt)
    legs_draw = torch.randint(2, max(cfg.looper_legs, 2) + 1, (n,), generator=gen, device=device)
    max_legs = torch.where(looper, legs_draw, torch.ones_like(legs_draw))
    charge = torch.where(rnd() < 0.5, -1.0, 1.0).to(torch.float64)
    eta = (2.0 * rnd() - 1.0) * cfg.eta_max
    eta = torch.where(looper, eta * (cfg.looper_eta_max / cfg.eta_max), eta)
    if cfg.one_side:
        eta = eta.abs()
    phi0 = cfg.az_lo * SECTOR_RAD + rnd() * (cfg.az_hi - cfg.az_lo) * SECTOR_RAD
    if cfg.len_law == "geometric":
        p = 1.0 / cfg.len_mean
        cap = torch.clamp(torch.floor(torch.log(1.0 - rnd()) / math.log(1.0 - p)) + 1.0, 1, 152).to(torch.int64)
    else:
        full = rnd() < cfg.full_len_frac
        cap = torch.where(full, torch.full((n,), 152, device=device),
                          torch.randint(cfg.len_lo, cfg.len_hi + 1, (n,), generator=gen, device=device))
    cap = torch.where(looper, 152 * max_legs, cap)
    row0 = torch.randint(0, cfg.row0_max + 1, (n,), generator=gen, device=device)
    t0 = torch.full((n,), 2000.0, **f64) if cfg.single_event else rnd() * (TF_NBINS - 500.0)
    z0 = 5.0 * torch.randn(n, generator=gen, **f64)

    kappa = charge * (KB_PER_TESLA * cfg.bz_tesla) / pt        # signed curvature, 1/cm
    circ = 2.0 * math.pi / kappa.abs()
    tanl = torch.sinh(eta)
    side = (eta < 0).to(torch.int64)
    az = torch.floor(phi0 / SECTOR_RAD).to(torch.int64) % 18
    az0 = az.clone()
    row_cur = row0 - 1
    dirn = torch.ones(n, dtype=torch.int64, device=device)
    leg = torch.zeros(n, dtype=torch.int64, device=device)
    s_prev = torch.zeros(n, **f64)
    alive = torch.ones(n, dtype=torch.bool, device=device)
    ncl = torch.zeros(n, dtype=torch.int64, device=device)
    miss = torch.zeros(n, dtype=torch.int64, device=device)
    last_hit = row0.clone()
    out = []
    S_MAX = 0.9
    for _ in range(152 * 6 + 128):
        idx = alive.nonzero(as_tuple=True)[0]
        if idx.numel() == 0:
            break
        cand = row_cur[idx] + dirn[idx]
        ex_out = cand > 151
        ex_in = cand < 0
        more = leg[idx] + 1 < max_legs[idx]
        kill = ex_out | (ex_in & ~more)
        alive[idx[kill]] = False
        flip = ex_in & more
        fi = idx[flip]
        leg[fi] += 1; dirn[fi] = 1; row_cur[fi] = -1; miss[fi] = 0
        az[fi] = az0[fi]
        keep = ~(kill | flip)
        idx = idx[keep]; cand = cand[keep]
        if idx.numel() == 0:
            continue
        xr = row_x[cand]
        k = kappa[idx]; ci = circ[idx]; sp_ = s_prev[idx]; d_ = dirn[idx]
        best_s = torch.full((idx.numel(),), float("inf"), **f64)
        best_y = torch.zeros(idx.numel(), **f64)
        best_az = torch.zeros(idx.numel(), dtype=torch.int64, device=device)
        for o in (0, 1, -1, 2, -2):
            a = (az[idx] + o) % 18
            p0 = phi0[idx] - (a.to(torch.float64) + 0.5) * SECTOR_RAD
            S = torch.sin(p0) + k * xr
            okS = S.abs() <= S_MAX
            asn = torch.asin(torch.clamp(S, -1.0, 1.0))
            pl = torch.where(d_ > 0, asn, math.pi - asn)
            s = torch.remainder((pl - p0) / k, ci)
            s = s + torch.ceil(torch.clamp_min(sp_ - s, 0.0) / ci) * ci
            s = torch.where(s <= sp_, s + ci, s)
            y = (torch.cos(p0) - torch.cos(pl)) / k
            good = okS & (y.abs() < half_w[cand]) & (s - sp_ < 0.6 * ci) & (s < best_s)
            if cfg.confine:
                good &= (a >= cfg.az_lo) & (a < cfg.az_hi)
            best_s = torch.where(good, s, best_s); best_y = torch.where(good, y, best_y); best_az = torch.where(good, a, best_az)
        found = torch.isfinite(best_s)
        z = z0[idx] + best_s * tanl[idx]
        found &= z.abs() < DRIFT_LEN_CM
        mi = idx[~found]
        miss[mi] += 1
        row_cur[mi] = cand[~found]
        too = miss[mi] > 6
        turn = too & (dirn[mi] > 0) & (leg[mi] + 1 < max_legs[mi])
        ti = mi[turn]
        leg[ti] += 1; dirn[ti] = -1; miss[ti] = 0; row_cur[ti] = last_hit[ti] + 1
        alive[mi[too & ~turn]] = False
        hi = idx[found]
        if hi.numel():
            r = cand[found]
            m = hi.numel()
            y = best_y[found] + cfg.noise_cm * torch.randn(m, generator=gen, **f64)
            zz = z[found] + cfg.noise_cm * torch.randn(m, generator=gen, **f64)
            uu = t0[hi] + (DRIFT_LEN_CM - zz.abs()) / DRIFT_CM_PER_BIN
            npd = npads[r]
            P = torch.minimum(torch.clamp_min(torch.round((y / padw[r] + npd / 2.0) * 64.0), 0.0), npd * 64 - 1).to(torch.int32)
            T = torch.clamp(torch.round(uu * 64.0), 0, (1 << 24) - 1).to(torch.int32)
            out.append((hi.to(torch.int32), leg[hi].to(torch.uint8), (side[hi] * 18 + best_az[found]).to(torch.uint8),
                        r.to(torch.uint8), P, T))
            az[hi] = best_az[found]; row_cur[hi] = r; last_hit[hi] = r; s_prev[hi] = best_s[found]; miss[hi] = 0
            ncl[hi] += 1
            alive[hi[ncl[hi] >= cap[hi]]] = False
    qpt = (kappa / (KB_PER_TESLA * cfg.bz_tesla)).to(torch.float32)
    if not out:
        e = torch.zeros(0, dtype=torch.int32, device=device)
        return (e, e.to(torch.uint8), e.to(torch.uint8), e.to(torch.uint8), e, e), ncl, qpt
    cols = [torch.cat(c) for c in zip(*out)]
    del out
    order = torch.sort(cols[0], stable=True).indices          # group by track, walk order kept inside the track
    return tuple(c[order] for c in cols), ncl, qpt


def generate_truth(cfg: EventConfig, geo: Geometry, device="cpu", batch: int = 400_000) -> Truth:
    """Attached-cluster truth of `cfg.n_tracks` tracks (the first tracks with >= cfg.min_ncl clusters, in draw order)."""
    device = torch.device(device)
    gen = torch.Generator(device=device)
    gen.manual_seed(cfg.seed)
    need = cfg.n_tracks
    parts = []
    while need > 0:
        n_draw = min(batch, int(need * 1.6) + 64)
        (tid, leg, sec, row, P, T), ncl, qpt = _trace(cfg, geo, gen, n_draw, device)
        good = (ncl >= cfg.min_ncl).nonzero(as_tuple=True)[0][:need]
        if good.numel() == 0:
            raise RuntimeError("no track survived; check the configuration")
        sel = torch.zeros(n_draw, dtype=torch.bool, device=device)
        sel[good] = True
        m = sel[tid.long()]
        n_att = int(m.sum())
        qtot, qmax, sigpad, sigtime, flags = _copy_through(gen, n_att, device)
        att = pack_records(T[m].long(), P[m].long(), qtot, qmax, sigpad, sigtime, flags, row[m].long(), sec[m].long())
        parts.append((ncl[good].to(torch.int16), qpt[good], att, leg[m]))
        need -= good.numel()
        del tid, leg, sec, row, P, T, m, sel
    return Truth(*(torch.cat(c) for c in zip(*parts)))


def generate_unattached_truth(geo: Geometry, n_unattached: int, seed: int, device="cpu", law: str = "inv_x",
                              single_event: bool = False) -> torch.Tensor:
    """Unattached clusters of one time frame in the CLUSTER domain (truth for an encoder; the encoder sorts
    them per region and stores differences).  Per-bin counts Poisson around the `law` density (total Poisson around
    n_unattached), pad uniform over the row's pads, time uniform over the time frame (or the event's 500 bins), in NO
    particular order inside a bin.  Returns int32 [n, 4] = 16-byte cluster records (layout.CLUSTER_DTYPE)."""
    device = torch.device(device)
    gen = torch.Generator(device=device)
    gen.manual_seed(seed * 7919 + 17)
    n_bins = geo.n_bins
    w = np.ones(n_bins) if law == "uniform" else np.tile(1.0 / geo.row_x_f64, geo.n_sectors_out)
    mean = torch.as_tensor(n_unattached * w / w.sum(), dtype=torch.float64, device=device)
    counts = torch.poisson(mean, generator=gen).to(torch.int64)
    n = int(counts.sum())
    bins = torch.repeat_interleave(torch.arange(n_bins, device=device), counts)
    bins = bins[torch.randperm(n, generator=gen, device=device)]                                # arbitrary order
    row = bins % geo.n_rows
    width = torch.as_tensor(geo.row_npads.astype(np.int64) * 64, device=device)[row]
    pad = (torch.rand(n, generator=gen, device=device, dtype=torch.float64) * width).to(torch.int64)
    span, base = (500.0 * 64.0, 2000.0 * 64.0) if single_event else (float(TF_NBINS) * 64.0, 0.0)
    time = (base + torch.rand(n, generator=gen, device=device, dtype=torch.float64) * span).to(torch.int64)
    qtot, qmax, sigpad, sigtime, flags = _copy_through(gen, n, device)
    return pack_records(time, pad, qtot, qmax, sigpad, sigtime, flags, row, bins // geo.n_rows)


# --- BASELINE.json configs at full size -----------------------------------------------------------------------------
WORKLOADS = {
    # name: (EventConfig factory, n_unattached, unattached single_event)
    "c1": (lambda: config1(10_000, 0, seed=2), 300_000, True),
    "c2": (lambda: config2_like(500_000, 0, seed=3), 20_000_000, False),
    "c3": (lambda: config2_like(2_000_000, 0, seed=4), 80_000_000, False),
    "c4": (lambda: config4_like(3_000_000, 0, seed=5), 30_000_000, False),
}
