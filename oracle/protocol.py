"""The paper's elongation protocol and the series of its tensile observables, fp64 numpy on
top of the C oracle's MD step.

TEST INFRASTRUCTURE ONLY, like the rest of oracle/: imported by tests/ alone; shares nothing with the CUDA path.

P:71: "The gripping atoms on the left and right sides of the wire are periodically displaced by 0.05 A in the [-100] and
[100] directions, respectively, between 20 ps of MD."  Both slabs are PLACED (reading A10): an atom of the
flag-2 slab sits at zref + D2, one of the flag-1 slab at zref + D1, with
    D(k) = disp0 + rate * k                      every step,           or
    D(k) = disp0 + rate * P * floor(k / P)       in strokes of P steps (paper: P = 10 000 steps of 2 fs, rate * P = 0.05 A),
k = steps of the run done, the current one included.
P:73: "ramping the temperature from 0.01 K to the target value": T(s) = T0 + T_rate * (s - step0), clamped at 0.
Eq.4: strain = (L - L0) / L0 with L - L0 = D2 - D1.  Eq.5 as read in DESIGN.md A11: observables.stress.
Rupture ("until rupture"): the wire has parted once the largest gap between consecutive z coordinates of its atoms
exceeds r_cut (no interaction crosses the gap any more).
Heat map (Fig.4): counts of (strain, stress) records of all replicas per cell of a regular grid.
"""
import numpy as np

from . import MD
from .observables import kinetic_tensor, stress


def slab_displacement(k, disp0, rate, period=0):
    """D(k), see the module header; k may be an array of step counts."""
    k = np.asarray(k, dtype=np.int64)
    if period and period > 0:
        k = (k // period) * period
    return np.asarray(disp0, dtype=np.float64) + np.asarray(rate, dtype=np.float64) * k


def temperature(T0, T_rate, steps_since_start):
    return np.maximum(np.asarray(T0, dtype=np.float64) + np.asarray(T_rate, dtype=np.float64) * steps_since_start, 0.0)


def largest_gap(z):
    """largest difference between consecutive values of z in sorted order"""
    zs = np.sort(np.asarray(z, dtype=np.float64))
    return float(np.max(np.diff(zs))) if len(zs) > 1 else 0.0


def heat_map(x, y, x_lo, x_hi, nx, y_lo, y_hi, ny):
    """counts[iy, ix] of the points with x in [x_lo, x_hi), y in [y_lo, y_hi); cell = floor((v - lo) / (hi - lo) * n)"""
    out = np.zeros((ny, nx), dtype=np.uint64)
    for xv, yv in zip(np.asarray(x, dtype=np.float64).ravel(), np.asarray(y, dtype=np.float64).ravel()):
        if not (x_lo <= xv < x_hi and y_lo <= yv < y_hi):
            continue
        ix = min(int(np.floor((xv - x_lo) / (x_hi - x_lo) * nx)), nx - 1)
        iy = min(int(np.floor((yv - y_lo) / (y_hi - y_lo) * ny)), ny - 1)
        out[iy, ix] += 1
    return out


class TensileMD:
    """oracle.MD driven by the protocol: two moving slabs, optional strokes, optional temperature ramp, and the series
    (step, strain, sigma_zz, largest z gap) recorded after every step s with (s + 1) % every == 0."""

    def __init__(self, md: MD, dt, T0, gamma, seed, step0, disp0_2, rate_2, disp0_1, rate_1, period=0, T_rate=None,
                 every=0, volume=None, L0=None, mass_amu=196.96657):
        self.md, self.dt, self.gamma, self.seed, self.step0 = md, dt, gamma, seed, int(step0)
        R = md.R
        b = lambda a: np.broadcast_to(np.asarray(0.0 if a is None else a, dtype=np.float64), (R,)).copy()
        self.T0, self.T_rate = b(T0), b(T_rate)
        self.d2, self.r2, self.d1, self.r1 = b(disp0_2), b(rate_2), b(disp0_1), b(rate_1)
        self.period, self.every = int(period), int(every)
        self.volume, self.L0, self.mass = b(volume), b(L0), mass_amu
        self.k = 0
        self.series = [[] for _ in range(R)]
        self.rupture_step = np.full(R, -1, dtype=np.int64)

    def step(self):
        md = self.md
        s = self.step0 + self.k                     # number of the step being taken
        D2 = slab_displacement(self.k + 1, self.d2, self.r2, self.period)
        D1 = slab_displacement(self.k + 1, self.d1, self.r1, self.period)
        T = temperature(self.T0, self.T_rate, self.k)
        # the flag-1 slab is placed here (orc_md_step leaves fixed atoms where they are), the flag-2 slab by orc_md_step
        for r in range(md.R):
            sl = slice(md.offsets[r], md.offsets[r + 1])
            f1 = md.flags[sl] == 1
            md.x[sl][f1, 2] = md.zref[sl][f1] + D1[r]
        md.step(self.dt, T, self.gamma, self.seed, s, slab_disp=D2)
        self.k += 1
        if self.every and (s + 1) % self.every == 0:
            K = kinetic_tensor(md.v, md.flags, md.offsets, self.mass)
            sig = stress(md.w_rep, K, self.volume)
            for r in range(md.R):
                sl = slice(md.offsets[r], md.offsets[r + 1])
                gap = largest_gap(md.x[sl, 2])
                self.series[r].append((float(s), (D2[r] - D1[r]) / self.L0[r], sig[r, 2], gap))
                if self.rupture_step[r] < 0 and gap > md.r_cut:
                    self.rupture_step[r] = s
