"""Nose-Hoover dynamics (the paper's thermostat) on top of the C oracle's forces, fp64 numpy.

TEST INFRASTRUCTURE ONLY, like the rest of oracle/: imported by tests/ alone; shares nothing with the CUDA path.

The paper says only "Nose-Hoover thermostat" (refs 39, 40) and gives neither the discretisation nor the
thermostat mass (reading A17).  Taken here: one thermostat variable xi per replica with
    d xi / dt = (2 K - g kB T) / Q,   d v / dt = F / m - xi v,   Q = g kB T tau^2,   g = 3 N_dyn,
integrated by the symmetric splitting  B A N A B  (kick, half drift, thermostat, half drift, [forces], kick) with
    N:  xi += (dt/2) (2 K - g kB T) / Q;   v *= s, s = exp(-xi dt);   K *= s^2;   xi += (dt/2) (2 K - g kB T) / Q,
K the kinetic energy of the dynamic atoms after the first kick.  xi = 0 and tau = infinity give velocity Verlet.
Conserved:  H' = E_pot + K + Q xi^2 / 2 + g kB T eta,  d eta / dt = xi  (eta advanced by the same N step:
eta += xi_mid dt with xi_mid the value used for the scaling).
Grips (flag != 0) are rigid and excluded from K (D:A12); this module does not move them.
"""
import numpy as np

from . import compute, au_params

KB = 8.617333262e-5
ACC = 9.648533212e-3


class NoseHooverMD:
    def __init__(self, x, v, flags, r_cut, T, tau_fs, lo=0.0, hi=0.0, periodic=0, offsets=None):
        self.prm = au_params()
        self.x = np.array(x, dtype=np.float64)
        self.v = np.array(v, dtype=np.float64)
        self.flags = np.asarray(flags)
        n = len(self.x)
        self.offsets = np.array([0, n], dtype=np.int32) if offsets is None else np.asarray(offsets, dtype=np.int32)
        self.R = len(self.offsets) - 1
        self.kw = dict(lo=lo, hi=hi, periodic=periodic, offsets=self.offsets)
        self.r_cut = r_cut
        self.T = np.broadcast_to(np.asarray(T, dtype=np.float64), (self.R,)).copy()
        self.tau = float(tau_fs)
        self.xi = np.zeros(self.R)
        self.eta = np.zeros(self.R)
        self.dyn = self.flags == 0
        self.g = np.array([3.0 * self.dyn[self.offsets[r]:self.offsets[r + 1]].sum() for r in range(self.R)])
        self.Q = self.g * KB * self.T * self.tau ** 2
        self.m = self.prm.mass_amu / ACC            # (m/c): energy = (m/c) v^2 / 2 in eV for v in A/fs
        o = compute(self.x, self.r_cut, **self.kw)
        self.f, self.e_rep = o["f"], o["e_rep"]

    def kinetic(self):
        return np.array([0.5 * self.m * np.sum(self.v[s][self.dyn[s]] ** 2) for s in self._slices()])

    def _slices(self):
        return [slice(self.offsets[r], self.offsets[r + 1]) for r in range(self.R)]

    def step(self, dt):
        kick = 0.5 * dt / self.m
        d = self.dyn[:, None]
        self.v = np.where(d, self.v + kick * self.f, 0.0)                  # B
        self.x = self.x + np.where(d, 0.5 * dt * self.v, 0.0)             # A
        K = self.kinetic()                                                # N
        for r, s in enumerate(self._slices()):
            gkt = self.g[r] * KB * self.T[r]
            self.xi[r] += 0.5 * dt * (2.0 * K[r] - gkt) / self.Q[r]
            sc = np.exp(-self.xi[r] * dt)
            self.eta[r] += self.xi[r] * dt
            self.v[s] *= sc
            self.xi[r] += 0.5 * dt * (2.0 * K[r] * sc * sc - gkt) / self.Q[r]
        self.x = self.x + np.where(d, 0.5 * dt * self.v, 0.0)             # A
        o = compute(self.x, self.r_cut, **self.kw)
        self.f, self.e_rep = o["f"], o["e_rep"]
        self.v = np.where(d, self.v + kick * self.f, 0.0)                  # B

    def conserved(self):
        return self.e_rep + self.kinetic() + 0.5 * self.Q * self.xi ** 2 + self.g * KB * self.T * self.eta
