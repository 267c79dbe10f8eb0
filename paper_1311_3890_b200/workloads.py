"""Seeded synthetic input generators (numpy only) -- shared by the oracle tests and the CUDA path.

This module holds NONE of the method's arithmetic (no energies, forces, neighbour predicates,
integrator or Philox): it only builds gold-nanowire / bulk geometries, Gaussian displacements,
Maxwell velocities and the per-replica metadata of the five BASELINE.json workloads.  It imports
neither `oracle` nor the CUDA binding.

The inputs stand in for the paper's own simulated wires (the paper uses no public dataset):
[100]-oriented cylindrical FCC Au nanowires (Fig. 1), two rigid gripping layers per
end, Gaussian initial velocities whose seed is the only difference between replicates
(P:71).  Recipe = DESIGN.md "Input recipe" (reading A13, A16).
"""
from dataclasses import dataclass, field

import numpy as np

A_LATTICE = 4.08          # Angstrom, BASELINE.json configs ("FCC a=4.08")
R_CUT = 7.0               # Angstrom, BASELINE.json configs
SKIN = 0.3                # Angstrom, BASELINE.json configs
MASS_AU = 196.96657       # amu
KB = 8.617333262e-5       # eV/K
ACC = 9.648533212e-3      # 1 eV/(A amu) in A/fs^2
DT_FS = 2.0
FLAG_DYNAMIC, FLAG_FIXED, FLAG_PULLED = 0, 1, 2


def fcc_wire(diameter, length, a=A_LATTICE):
    """[100]||z cylindrical FCC wire (reading A16): conventional cells, axis through a lattice
    point, keep x^2+y^2 <= (D/2)^2 + 1e-9, n_z = round(L/a) cells = 2 n_z (100) layers, z centred
    on 0.  Atoms are ordered along the wire axis, layer by layer.  Returns (n,3) float64."""
    rad2 = (0.5 * diameter) ** 2 + 1e-9
    nz = int(round(length / a))
    m = int(np.ceil(0.5 * diameter / a)) + 1
    basis = np.array([[0, 0, 0], [0.5, 0.5, 0], [0.5, 0, 0.5], [0, 0.5, 0.5]])
    ix, iy, iz = np.meshgrid(np.arange(-m, m + 1), np.arange(-m, m + 1), np.arange(nz), indexing="ij")
    cells = np.stack([ix.ravel(), iy.ravel(), iz.ravel()], axis=1).astype(np.float64)
    pts = (cells[:, None, :] + basis[None, :, :]).reshape(-1, 3) * a
    pts = pts[pts[:, 0] ** 2 + pts[:, 1] ** 2 <= rad2]
    order = np.lexsort((pts[:, 0], pts[:, 1], pts[:, 2]))   # z-major: ordered along [100]
    pts = pts[order]
    pts[:, 2] -= 0.5 * (pts[:, 2].min() + pts[:, 2].max())
    return pts


def ring_notch(x, a=A_LATTICE, planes=3, per_plane=9):
    """The paper's "small, ring-shaped notch ... in the center of the NW ... three atoms wide and two atoms deep" (P:71,
    P:77), reading A18: from each of the `planes` (100) planes nearest the wire's centre the `per_plane` atoms farthest
    from the axis are removed (ties by azimuth): with 9 that is the two outermost radial shells of a 3.1 nm wire and
    27 atoms in all, the difference between 8 850 and the 8 823 atoms of Table 2's first row.  Returns the
    remaining atoms, order kept."""
    z = x[:, 2]
    lev_of = np.round((z - z.min()) / (0.5 * a)).astype(np.int64)      # (100) planes are a / 2 apart
    levels = np.unique(lev_of)
    zc = 0.5 * (z.min() + z.max())
    centre = levels[np.argsort(np.abs(z.min() + levels * 0.5 * a - zc), kind="stable")[:planes]]
    r = np.hypot(x[:, 0], x[:, 1])
    phi = np.arctan2(x[:, 1], x[:, 0])
    keep = np.ones(len(x), bool)
    for lv in centre:
        idx = np.nonzero(lev_of == lv)[0]
        order = idx[np.lexsort((phi[idx], -np.round(r[idx], 6)))]
        keep[order[:per_plane]] = False
    return x[keep]


def fcc_bulk(ncell, a=A_LATTICE):
    """Periodic cubic FCC block of ncell^3 conventional cells in [0, ncell*a)^3, z-major order."""
    basis = np.array([[0, 0, 0], [0.5, 0.5, 0], [0.5, 0, 0.5], [0, 0.5, 0.5]])
    iz, iy, ix = np.meshgrid(np.arange(ncell), np.arange(ncell), np.arange(ncell), indexing="ij")
    cells = np.stack([ix.ravel(), iy.ravel(), iz.ravel()], axis=1).astype(np.float64)
    return (cells[:, None, :] + basis[None, :, :]).reshape(-1, 3) * a


def displace(x, sigma, seed):
    """Add seeded N(0, sigma^2) displacements per component."""
    rng = np.random.default_rng(seed)
    return x + rng.normal(0.0, sigma, size=x.shape)


def grip_flags(x, n_layers=2, a=A_LATTICE):
    """Two outermost (100) planes (spacing a/2) at each end are rigid (reading A12):
    bottom end fixed (flag 1), top end pulled (flag 2)."""
    z = x[:, 2]
    tol = 0.25 * a
    flags = np.zeros(len(x), dtype=np.int32)
    flags[z < z.min() + (n_layers - 1) * 0.5 * a + tol] = FLAG_FIXED
    flags[z > z.max() - (n_layers - 1) * 0.5 * a - tol] = FLAG_PULLED
    return flags


def maxwell_velocities(n, T, seed, dynamic=None, mass=MASS_AU):
    """Gaussian velocities (A/fs) at temperature T from a seed ("random Gaussian distribution
    of atomic velocities"; reading A13): N(0, kB T c/m) per component, centre-of-mass velocity of
    the dynamic atoms removed, then rescaled so that sum (m/2c) v^2 = (3/2)(N_dyn - 1) kB T.
    Non-dynamic atoms get v = 0."""
    rng = np.random.default_rng(seed)
    dyn = np.ones(n, dtype=bool) if dynamic is None else np.asarray(dynamic, dtype=bool)
    v = rng.normal(0.0, np.sqrt(KB * T * ACC / mass), size=(n, 3))
    v[~dyn] = 0.0
    nd = int(dyn.sum())
    if nd > 1 and T > 0:
        v[dyn] -= v[dyn].mean(axis=0)
        ek = 0.5 * mass / ACC * np.sum(v[dyn] ** 2)
        v[dyn] *= np.sqrt(1.5 * (nd - 1) * KB * T / ek)
    return v


def pack_pos4(x, flags=None):
    """(n,3) float64 -> (n,4) float32 with w = flag bits as an int32 bit pattern."""
    p = np.zeros((len(x), 4), dtype=np.float32)
    p[:, :3] = x
    if flags is not None:
        p[:, 3] = np.asarray(flags, dtype=np.int32).view(np.float32)
    return p


def pack_vel4(v, x32, flags=None):
    """(n,3) -> (n,4) float32 with w = reference z of the atom (used for grip atoms: a pulled
    atom is placed at w + D_r)."""
    q = np.zeros((len(v), 4), dtype=np.float32)
    q[:, :3] = v
    q[:, 3] = x32[:, 2]
    return q


@dataclass
class Workload:
    """One batch of independent replicas.  Arrays are host numpy; positions are fp32-exact."""
    name: str
    pos4: np.ndarray            # (N,4) float32, w = flags
    vel4: np.ndarray            # (N,4) float32, w = z_ref
    offsets: np.ndarray         # (R+1,) int32
    box_lo: np.ndarray          # (R,3) float32
    box_hi: np.ndarray          # (R,3) float32
    periodic: np.ndarray        # (R,3) uint8
    T: np.ndarray               # (R,) float32  thermostat temperature
    seed: np.ndarray            # (R,) uint64   Philox key
    slab_rate: np.ndarray       # (R,) float64  pulled-slab displacement per step, Angstrom
    gamma: float = 0.0          # 1/fs
    dt: float = DT_FS
    r_cut: float = R_CUT
    skin: float = SKIN
    rebuild_every: int = 0      # 0 = displacement-triggered (reading A14)
    meta: dict = field(default_factory=dict)

    @property
    def n_atoms(self):
        return int(self.offsets[-1])

    @property
    def n_replicas(self):
        return len(self.offsets) - 1

    @property
    def flags(self):
        return self.pos4[:, 3].view(np.int32)

    def x64(self):
        return self.pos4[:, :3].astype(np.float64)

    def v64(self):
        return self.vel4[:, :3].astype(np.float64)

    def take(self, r0, r1, name=None):
        """Sub-batch of replicas [r0, r1) (used for sharding across ranks and bounded CPU samples)."""
        a0, a1 = int(self.offsets[r0]), int(self.offsets[r1])
        return Workload(name or f"{self.name}[{r0}:{r1}]", self.pos4[a0:a1].copy(), self.vel4[a0:a1].copy(),
                        (self.offsets[r0:r1 + 1] - a0).astype(np.int32), self.box_lo[r0:r1].copy(),
                        self.box_hi[r0:r1].copy(), self.periodic[r0:r1].copy(), self.T[r0:r1].copy(),
                        self.seed[r0:r1].copy(), self.slab_rate[r0:r1].copy(), self.gamma, self.dt,
                        self.r_cut, self.skin, self.rebuild_every, dict(self.meta))


def _wire_box(x, pad_xy=2.0, pad_z=2.0, stretch=0.0):
    lo = x.min(axis=0) - np.array([pad_xy, pad_xy, pad_z])
    hi = x.max(axis=0) + np.array([pad_xy, pad_xy, pad_z + stretch])
    return lo, hi


def _assemble(name, wires, flags, vels, T, seeds, rates, gamma, stretch=0.0, **kw):
    offs = np.zeros(len(wires) + 1, dtype=np.int32)
    offs[1:] = np.cumsum([len(w) for w in wires])
    x = np.concatenate(wires)
    fl = np.concatenate(flags)
    pos4 = pack_pos4(x, fl)
    vel4 = pack_vel4(np.concatenate(vels), pos4, fl)
    lo = np.zeros((len(wires), 3), dtype=np.float32)
    hi = np.zeros((len(wires), 3), dtype=np.float32)
    for r, w in enumerate(wires):
        l, h = _wire_box(w, stretch=stretch)
        lo[r], hi[r] = l, h
    per = np.zeros((len(wires), 3), dtype=np.uint8)
    return Workload(name, pos4, vel4, offs, lo, hi, per, np.asarray(T, dtype=np.float32),
                    np.asarray(seeds, dtype=np.uint64), np.asarray(rates, dtype=np.float64), gamma, **kw)


STRAIN_RATE_PER_FS = 1e8 * 1e-15   # 1e8 1/s (BASELINE.json configs 2-4)


def config1(seed=1):
    """BASELINE config 1: one 3 nm x 6 nm wire, sigma = 0.05 A displacements, non-periodic,
    v = 0, NVE (gamma = 0), no grips.  N = 2655."""
    x = displace(fcc_wire(30.0, 60.0), 0.05, seed)
    n = len(x)
    return _assemble("config1_wire_3x6nm", [x], [np.zeros(n, np.int32)], [np.zeros((n, 3))],
                     [0.0], [seed], [0.0], 0.0, meta=dict(config=1))


def config2(seed=2, diameter=30.0, length=120.0, T=298.0):
    """BASELINE config 2: one 3 nm x 12 nm wire, 2 rigid (100) layers per end, Maxwell 298 K,
    Langevin gamma = 1/ps, top slab pulled at strain rate 1e8 1/s.  N = 5133."""
    x = fcc_wire(diameter, length)
    fl = grip_flags(x)
    v = maxwell_velocities(len(x), T, seed, fl == 0)
    L0 = x[:, 2].max() - x[:, 2].min()
    return _assemble("config2_wire_3x12nm_langevin_pull", [x], [fl], [v], [T], [seed],
                     [STRAIN_RATE_PER_FS * L0 * DT_FS], 1e-3, stretch=0.05 * L0, meta=dict(config=2))


def _replica_batch(name, n_rep, diameter, length, temps, seed0, jitter_layers=False, cfg=0):
    base = fcc_wire(diameter, length)
    layer_z = np.unique(np.round(base[:, 2], 6))
    rng = np.random.default_rng(seed0)
    wires, flags, vels, seeds, rates = [], [], [], [], []
    variants = {}
    for r in range(n_rep):
        dl = int(rng.integers(-1, 2)) if jitter_layers else 0
        if dl not in variants:
            if dl == 0:
                xv = base
            elif dl < 0:                       # drop the top layer
                xv = base[base[:, 2] < layer_z[-1] - 1e-6].copy()
            else:                              # one more layer = a longer wire cut back by one layer
                longer = fcc_wire(diameter, length + A_LATTICE)
                lz = np.unique(np.round(longer[:, 2], 6))
                xv = longer[longer[:, 2] < lz[-1] - 1e-6].copy()
            xv = xv.copy()
            xv[:, 2] -= 0.5 * (xv[:, 2].min() + xv[:, 2].max())
            variants[dl] = (xv, grip_flags(xv))
        xv, fl = variants[dl]
        s = seed0 * 100003 + r
        wires.append(xv)
        flags.append(fl)
        vels.append(maxwell_velocities(len(xv), temps[r], s, fl == 0))
        seeds.append(s)
        L0 = xv[:, 2].max() - xv[:, 2].min()
        rates.append(STRAIN_RATE_PER_FS * L0 * DT_FS)
    L0 = base[:, 2].max() - base[:, 2].min()
    return _assemble(name, wires, flags, vels, temps, seeds, rates, 1e-3, stretch=0.05 * L0,
                     meta=dict(config=cfg))


def config3(n_rep=256, seed=3, length=240.0):
    """BASELINE config 3: 256 replicas of a 3 nm x 24 nm wire (10 443 atoms each), replicas
    [0, R/2) at 10 K and [R/2, R) at 298 K, own seed/box each, Langevin + pulling."""
    temps = [10.0 if r < n_rep // 2 else 298.0 for r in range(n_rep)]
    return _replica_batch(f"config3_{n_rep}x_wire_3x24nm", n_rep, 30.0, length, temps, seed, cfg=3)


def config4(n_rep=2048, seed=4):
    """BASELINE config 4: 2048 replicas of 3 nm x 6 nm wires, number of (100) layers jittered by
    U{-1,0,+1} per replica from the seed, 298 K Langevin + pulling."""
    return _replica_batch(f"config4_{n_rep}x_wire_3x6nm_jitter", n_rep, 30.0, 60.0, [298.0] * n_rep,
                          seed, jitter_layers=True, cfg=4)


def paper_wire(k=1, T=10.0, n_rep=1, seed=7):
    """The shapes of the paper's own benchmark (Table 2): unstretched [100] Au wires of
    D0 = 3.1 nm and L0 = 20.4 k nm (8 850 k atoms; the paper's sizes are 8 823 + 8 850 (k - 1), with a 27-atom notch that
    is left out here), r_cut = 5.8 A, buffer 0.29 A, dt = 2 fs, at 10 K or 298 K, not pulled.  The paper's
    thermostat is Nose-Hoover; Langevin (gamma = 1/ps) stands in for it.  n_rep > 1 batches identical wires with their own
    seeds (the paper runs one per GPU)."""
    x = fcc_wire(31.0, 204.0 * k)
    fl = np.zeros(len(x), np.int32)
    wires, flags, vels, seeds = [], [], [], []
    for r in range(n_rep):
        s = seed * 100003 + r
        wires.append(x); flags.append(fl); seeds.append(s)
        vels.append(maxwell_velocities(len(x), T, s, fl == 0))
    w = _assemble(f"paper_table2_{n_rep}x_wire_3.1x{20.4 * k:.1f}nm_{T:g}K", wires, flags, vels, [T] * n_rep, seeds,
                  [0.0] * n_rep, 1e-3, meta=dict(config="paper", k=k))
    w.r_cut = 5.8
    w.skin = 0.29
    return w


def config5a(ncell=64, seed=5):
    """BASELINE config 5 (bulk): periodic FCC ncell^3 cells, sigma = 0.05 A displacements,
    NVE, neighbour rebuild every 10 steps.  ncell = 64 -> 1 048 576 atoms."""
    L = ncell * A_LATTICE
    x = displace(fcc_bulk(ncell), 0.05, seed)
    x32 = x.astype(np.float32)
    Lf = np.float32(L)
    x32 = np.where(x32 < 0, x32 + Lf, x32)
    x32 = np.where(x32 >= Lf, x32 - Lf, x32).astype(np.float32)   # wrapped into [0, L) in fp32
    n = len(x32)
    pos4 = pack_pos4(x32, np.zeros(n, np.int32))
    vel4 = pack_vel4(np.zeros((n, 3)), pos4)
    return Workload(f"config5a_bulk_{ncell}cubed", pos4, vel4, np.array([0, n], np.int32),
                    np.zeros((1, 3), np.float32), np.full((1, 3), L, np.float32),
                    np.ones((1, 3), np.uint8), np.zeros(1, np.float32), np.array([seed], np.uint64),
                    np.zeros(1), 0.0, rebuild_every=10, meta=dict(config=5))


def config5b(seed=6, diameter=60.0, length=1000.0):
    """BASELINE config 5 (wire): one 6 nm x 100 nm wire (164 885 atoms), sigma = 0.05 A, NVE,
    rebuild every 10 steps."""
    x = displace(fcc_wire(diameter, length), 0.05, seed)
    n = len(x)
    w = _assemble("config5b_wire_6x100nm", [x], [np.zeros(n, np.int32)], [np.zeros((n, 3))], [0.0],
                  [seed], [0.0], 0.0, meta=dict(config=5))
    w.rebuild_every = 10
    return w
