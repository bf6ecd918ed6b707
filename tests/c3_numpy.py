"""A second, independent evaluation of the attached-cluster track model: numpy float32 SCALARS, written from the op list
SURVEY.md §8(c)-C3 (lines 356-394) and the readings of DESIGN.md §3 -- not from oracle/tmd_oracle.c.

It is the pin SURVEY.md §8(c)-C8 row 2 asks for ("a second, independent oracle-side implementation in numpy float32
scalars (numpy never fuses) compared ... incl. all per-step states").  It imports nothing from oracle/ and nothing from
the CUDA package; the geometry tables come in as inputs, exactly as they do for the oracle and the library.

Every arithmetic step is one numpy float32 scalar operation (IEEE-754 binary32, round to nearest even; numpy does not
contract a*b+c).  Paper passages: PAPER.md L70 ("propagates it through the TPC and computes the absolute values of the
coordinates using the residuals given in input and the reconstructed track"), L68 (residual to the track).
"""
from __future__ import annotations

import numpy as np

F = np.float32
ONE, HALF, QUARTER = F(1.0), F(0.5), F(0.25)
SP_MAX, S_MIN, DT_MAX = F(0.95), F(0.001), F(8.0)
INV64, SIXTYFOUR = F(0.015625), F(64.0)
C24 = np.array([0x3D2AAAAB], np.uint32).view(np.float32)[0]          # fp32(1/24), C1
LIGHT = F(0.00299792458)
P_MAX, T_MAX = F(65535.0), F(16777215.0)

COLUMNS = ("sec", "row", "dir", "ok", "x", "y", "sp", "sp2", "y2", "u2", "s", "P_pred", "T_pred", "P", "T",
           "yn", "un", "spn", "dtn", "kn")
FLOAT_COLUMNS = ("x", "y", "sp", "sp2", "y2", "u2", "s", "yn", "un", "spn", "dtn", "kn")
ONLY_IF_OK = ("y2", "u2", "s")                                        # C3-6: "If !ok, none of cp1..u2 is used"


def bits(v) -> int:
    return int(np.array([v], np.float32).view(np.uint32)[0])


def clamp(v, lo, hi):
    """fminf(fmaxf(v, lo), hi): np.fmax / np.fmin return the non-NaN operand, so NaN -> lo."""
    return F(np.fmin(np.fmax(F(v), F(lo)), F(hi)))


class Model:
    def __init__(self, geo, bz_tesla: float):
        self.n_az, self.n_rows = int(geo.n_az), int(geo.n_rows)
        self.cos_a, self.sin_a = F(geo.cos_a), F(geo.sin_a)
        self.row_x = np.asarray(geo.row_x, np.float32)
        self.padw = np.asarray(geo.row_padw, np.float32)
        self.inv_padw = np.asarray(geo.row_inv_padw, np.float32)
        self.half = (np.asarray(geo.row_npads).astype(np.int64) // 2).astype(np.float32)
        kb = F(F(bz_tesla) * LIGHT)                                   # KB, C1
        self.qk = F(F(0.0625) * kb)                                   # QK, C1

    # ---- helpers (C3 "Helpers")
    def pad2y(self, r: int, P: int):
        return F(F(F(F(np.uint32(P)) * INV64) - self.half[r]) * self.padw[r])

    @staticmethod
    def time2u(T: int):
        return F(F(np.uint32(T)) * INV64)

    def quantP(self, y, r: int) -> int:
        pf = F(F(y * self.inv_padw[r]) + self.half[r])
        v = np.floor(F(F(pf * SIXTYFOUR) + HALF))
        return int(clamp(v, F(0.0), P_MAX))

    @staticmethod
    def quantT(u) -> int:
        v = np.floor(F(F(u * SIXTYFOUR) + HALF))
        return int(clamp(v, F(0.0), T_MAX))

    # ---- C3-1, C3-2
    def init(self, qpt: int, row0: int, P0: int, T0: int) -> dict:
        k = F(F(np.int8(qpt)) * self.qk)
        x = self.row_x[row0]
        y = self.pad2y(row0, P0)
        u = self.time2u(T0)
        L = np.sqrt(F(F(x * x) + F(y * y)))
        sd = clamp(F(F(HALF * k) * L), -SP_MAX, SP_MAX)
        cd = np.sqrt(F(ONE - F(sd * sd)))
        sp = clamp(F(F(F(y * cd) + F(x * sd)) / L), -SP_MAX, SP_MAX)
        return dict(x=x, y=y, u=u, sp=sp, dt=F(0.0), k=k, dir=+1)

    # ---- C3-3 .. C3-9 for cluster j >= 1; returns the trace row (bit patterns for the float columns)
    def step(self, st: dict, sec: int, row: int, P_prev: int, T_prev: int, j: int, rowdiff: int, secleg: int,
             padres: int, timeres: int):
        x, y, u, sp, dt, k, dirn = st["x"], st["y"], st["u"], st["sp"], st["dt"], st["k"], st["dir"]
        n_rows, n_az = self.n_rows, self.n_az
        # C3-3 leg
        if secleg & 0x80:
            dirn, sp, dt, k = -dirn, F(-sp), F(-dt), F(-k)
        # C3-4 row (reading 19: the stored byte is reduced mod n_rows first)
        rd = rowdiff % n_rows
        row = (row + (rd if dirn > 0 else n_rows - rd)) % n_rows
        # C3-5 sector (reading 19: bit 6 ignored, the step reduced mod n_az; the side never changes)
        d = (secleg & 0x3F) % n_az
        if d != 0:
            az, side = sec % n_az, sec // n_az
            sec = side * n_az + (az + d) % n_az
            steps = d if d <= n_az // 2 else d - n_az
            sn = self.sin_a if steps > 0 else F(-self.sin_a)
            for _ in range(abs(steps)):
                cp = np.sqrt(F(ONE - F(sp * sp)))
                xn = F(F(x * self.cos_a) + F(y * sn))
                yn = F(F(y * self.cos_a) - F(x * sn))
                spn = clamp(F(F(sp * self.cos_a) - F(cp * sn)), -SP_MAX, SP_MAX)
                x, y, sp = xn, yn, spn
        tr = dict(sec=sec, row=row, dir=dirn, x=bits(x), y=bits(y), sp=bits(sp))
        # C3-6 propagate
        xt = self.row_x[row]
        dx = F(xt - x)
        sp2 = F(sp + F(k * dx))
        ok = not (np.abs(sp2) > SP_MAX)
        y2 = u2 = s = None
        if ok:
            cp1 = np.sqrt(F(ONE - F(sp * sp)))
            cp2 = np.sqrt(F(ONE - F(sp2 * sp2)))
            dy = F(F(dx * F(sp + sp2)) / F(cp1 + cp2))
            ch = np.sqrt(F(F(dx * dx) + F(dy * dy)))
            if dx < 0:
                ch = F(-ch)
            kc = F(k * ch)
            s = F(ch * F(ONE + F(F(kc * kc) * C24)))
            y2 = F(y + dy)
            u2 = F(u + F(dt * s))
            P_pred, T_pred = self.quantP(y2, row), self.quantT(u2)      # C3-7
        else:
            P_pred, T_pred = P_prev, T_prev                             # reading 8
        # C3-8 rebuild
        P = (P_pred + padres) & 0xFFFF
        T = (T_pred + timeres) & 0xFFFFFFFF
        # C3-9 update
        ym, um = self.pad2y(row, P), self.time2u(T)
        if not ok:
            y, u, sp = ym, um, clamp(sp2, -SP_MAX, SP_MAX)
        else:
            ry, ru = F(ym - y2), F(um - u2)
            y = F(y2 + F(HALF * ry))
            u = F(u2 + F(HALF * ru))
            if np.abs(s) >= S_MIN:
                sp = clamp(F(sp2 + F(F(QUARTER * ry) / s)), -SP_MAX, SP_MAX)
                bu = ONE if j == 1 else QUARTER
                dt = clamp(F(dt + F(F(bu * ru) / s)), -DT_MAX, DT_MAX)
            else:
                sp = clamp(sp2, -SP_MAX, SP_MAX)
        st.update(x=xt, y=y, u=u, sp=sp, dt=dt, k=k, dir=dirn)
        tr.update(ok=int(ok), sp2=bits(sp2), y2=bits(y2) if ok else None, u2=bits(u2) if ok else None,
                  s=bits(s) if ok else None, P_pred=P_pred, T_pred=T_pred, P=P, T=T,
                  yn=bits(y), un=bits(u), spn=bits(sp), dtn=bits(dt), kn=bits(k))
        return tr, sec, row, P, T

    def decode_track(self, qpt: int, sec0: int, row0: int, P0: int, T0: int, rowdiff, secleg, padres, timeres):
        """-> dict(sec, row, P, T lists of ncl entries; trace rows for j = 1..ncl-1; init and final state bits (x,y,u,sp,dt,k))."""
        with np.errstate(all="ignore"):                                 # NaN / inf are defined results here (reading 15)
            st = self.init(qpt, row0, P0, T0)
            state_bits = lambda: [bits(st[c]) for c in ("x", "y", "u", "sp", "dt", "k")]
            out = dict(sec=[sec0], row=[row0], P=[P0 & 0xFFFF], T=[T0 & 0xFFFFFFFF], trace=[], init=state_bits())
            sec, row, P, T = sec0, row0, P0 & 0xFFFF, T0 & 0xFFFFFFFF
            for j in range(1, len(rowdiff) + 1):
                tr, sec, row, P, T = self.step(st, sec, row, P, T, j, int(rowdiff[j - 1]), int(secleg[j - 1]),
                                               int(padres[j - 1]) & 0xFFFF, int(timeres[j - 1]) & 0xFFFFFFFF)
                out["trace"].append(tr)
                for key, v in (("sec", sec), ("row", row), ("P", P), ("T", T)):
                    out[key].append(v)
            out["final"] = state_bits()
        return out


def same_bits(a: int, b: int) -> bool:
    """Equal bit patterns, or both NaN (payloads / signs of NaN are not compared: DESIGN.md §3 reading 15)."""
    if a == b:
        return True
    isnan = lambda w: (w & 0x7F800000) == 0x7F800000 and (w & 0x007FFFFF) != 0
    return isnan(a) and isnan(b)
