"""ctypes front end of the fp64 CPU oracle (oracle/tbsma_oracle.c).

TEST INFRASTRUCTURE ONLY: imported by tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs.  Never imported by paper_1311_3890_b200 (the product),
and it imports nothing from it.  Every function is a thin marshalling layer; all arithmetic
is in the C file, which cites the paper line by line (the observables of P:79-87 -- kinetic
tensor, virial stress, strain -- are plain numpy in oracle/observables.py, and the paper's
Nose-Hoover thermostat in oracle/nose_hoover.py on top of this module's forces).
"""
import ctypes as C
import os

import numpy as np

from .build import build as _build

_lib = None


class Params(C.Structure):
    """Table 1 of the paper with r0 read as a/sqrt(2) (reading A1)."""
    _fields_ = [("A", C.c_double), ("xi", C.c_double), ("p", C.c_double),
                ("q", C.c_double), ("r0", C.c_double), ("mass_amu", C.c_double)]


def au_params() -> Params:
    return Params(0.2061, 1.790, 10.229, 4.036, 2.884, 196.96657)


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build())
        _lib.orc_num_threads.restype = C.c_int
    return _lib


def num_threads() -> int:
    return int(lib().orc_num_threads())


def _p(a, t):
    return None if a is None else a.ctypes.data_as(C.POINTER(t))


def _topo(n, offsets, lo, hi, periodic):
    if offsets is None:
        offsets = np.array([0, n], dtype=np.int32)
    offsets = np.ascontiguousarray(offsets, dtype=np.int32)
    R = len(offsets) - 1
    lo = np.ascontiguousarray(np.broadcast_to(np.asarray(lo, dtype=np.float32), (R, 3)))
    hi = np.ascontiguousarray(np.broadcast_to(np.asarray(hi, dtype=np.float32), (R, 3)))
    per = np.ascontiguousarray(np.broadcast_to(np.asarray(periodic, dtype=np.uint8), (R, 3)))
    return R, offsets, lo, hi, per


def neighbors(pos4, radius, offsets=None, lo=0.0, hi=0.0, periodic=0, max_nb=128):
    """Brute-force neighbour sets by predicate A6.  Returns (counts[n], list[n,max_nb])."""
    pos4 = np.ascontiguousarray(pos4, dtype=np.float32)
    n = pos4.shape[0]
    R, offsets, lo, hi, per = _topo(n, offsets, lo, hi, periodic)
    counts = np.zeros(n, dtype=np.int32)
    lst = np.full((n, max_nb), -1, dtype=np.int32)
    mx = lib().orc_neighbors(C.c_int64(n), _p(pos4, C.c_float), C.c_int32(R), _p(offsets, C.c_int32),
                             _p(lo, C.c_float), _p(hi, C.c_float), _p(per, C.c_uint8),
                             C.c_double(radius), C.c_int32(max_nb), _p(counts, C.c_int32),
                             _p(lst, C.c_int32))
    if mx < 0 or mx > max_nb:
        raise RuntimeError(f"oracle neighbors: max count {mx} exceeds max_nb {max_nb}")
    return counts, lst


def compute(x, r_cut, params=None, offsets=None, lo=0.0, hi=0.0, periodic=0, fp32_pred=True,
            cells=False):
    """Energies, forces, virial by brute force (cells=True: the linked-cell path).

    x: (n,3) float64.  Returns dict(rho, e_atom, f, e_rep, w_rep[, n_pairs_directed])."""
    params = params or au_params()
    x = np.ascontiguousarray(x, dtype=np.float64)
    n = x.shape[0]
    R, offsets, lo, hi, per = _topo(n, offsets, lo, hi, periodic)
    out = dict(rho=np.zeros(n), e_atom=np.zeros(n), f=np.zeros((n, 3)), e_rep=np.zeros(R),
               w_rep=np.zeros((R, 6)))
    d = C.c_double
    common = [C.byref(params), d(r_cut), C.c_int64(n), _p(x, d), C.c_int32(R), _p(offsets, C.c_int32),
              _p(lo, C.c_float), _p(hi, C.c_float), _p(per, C.c_uint8), C.c_int(int(fp32_pred)),
              _p(out["rho"], d), _p(out["e_atom"], d), _p(out["f"], d), _p(out["e_rep"], d),
              _p(out["w_rep"], d)]
    if cells:
        npairs = C.c_int64(0)
        rc = lib().orc_compute_celllist(*common, C.byref(npairs))
        out["n_pairs_directed"] = int(npairs.value)
    else:
        rc = lib().orc_compute(*common)
    if rc != 0:
        raise RuntimeError(f"oracle compute failed rc={rc}")
    return out


def compute_sample(x, r_cut, idx, params=None, offsets=None, lo=0.0, hi=0.0, periodic=0,
                   fp32_pred=True):
    """rho, E_i, F_i of the atoms idx, each from scratch by brute force (full-size parity)."""
    params = params or au_params()
    x = np.ascontiguousarray(x, dtype=np.float64)
    n = x.shape[0]
    R, offsets, lo, hi, per = _topo(n, offsets, lo, hi, periodic)
    idx = np.ascontiguousarray(idx, dtype=np.int64)
    rep = (np.searchsorted(offsets, idx, side="right") - 1).astype(np.int32)
    m = len(idx)
    out = dict(rho=np.zeros(m), e_atom=np.zeros(m), f=np.zeros((m, 3)))
    d = C.c_double
    rc = lib().orc_compute_sample(C.byref(params), d(r_cut), _p(x, d), _p(offsets, C.c_int32),
                                  _p(lo, C.c_float), _p(hi, C.c_float), _p(per, C.c_uint8),
                                  C.c_int(int(fp32_pred)), C.c_int64(m), _p(idx, C.c_int64),
                                  _p(rep, C.c_int32), _p(out["rho"], d), _p(out["e_atom"], d),
                                  _p(out["f"], d))
    if rc != 0:
        raise RuntimeError(f"oracle compute_sample failed rc={rc}")
    return out


def philox4x32_10(ctr, key):
    ctr = np.ascontiguousarray(ctr, dtype=np.uint32)
    key = np.ascontiguousarray(key, dtype=np.uint32)
    out = np.zeros(4, dtype=np.uint32)
    lib().orc_philox4x32_10(_p(ctr, C.c_uint32), _p(key, C.c_uint32), _p(out, C.c_uint32))
    return out


def gauss3(seed, tag, step):
    g = np.zeros(3)
    raw = np.zeros(4, dtype=np.uint32)
    lib().orc_gauss3(C.c_uint64(seed), C.c_uint32(tag), C.c_uint64(step), _p(g, C.c_double),
                     _p(raw, C.c_uint32))
    return g, raw


class MD:
    """State holder around orc_md_step (BAOAB / velocity Verlet, grips; reading A8, A12)."""

    def __init__(self, x, v, flags, r_cut, params=None, offsets=None, lo=0.0, hi=0.0, periodic=0,
                 fp32_pred=False, cells=False, zref=None):
        self.params = params or au_params()
        self.x = np.array(x, dtype=np.float64, order="C")
        self.v = np.array(v, dtype=np.float64, order="C")
        self.n = self.x.shape[0]
        self.flags = np.ascontiguousarray(flags, dtype=np.int32)
        self.zref = np.array(self.x[:, 2] if zref is None else zref, dtype=np.float64, order="C")
        self.r_cut = float(r_cut)
        self.R, self.offsets, self.lo, self.hi, self.per = _topo(self.n, offsets, lo, hi, periodic)
        self.fp32_pred = int(fp32_pred)
        self.cells = int(cells)
        self.rho = np.zeros(self.n)
        self.e_atom = np.zeros(self.n)
        self.e_rep = np.zeros(self.R)
        self.w_rep = np.zeros((self.R, 6))
        self.ekin_rep = np.zeros(self.R)
        out = compute(self.x, self.r_cut, self.params, self.offsets, self.lo, self.hi, self.per,
                      bool(fp32_pred), cells=bool(cells))
        self.f = out["f"]
        self.e_rep[:] = out["e_rep"]
        self.w_rep[:] = out["w_rep"]
        m = self.params.mass_amu / 9.648533212e-3
        dyn = self.flags == 0
        for r in range(self.R):
            s = slice(self.offsets[r], self.offsets[r + 1])
            self.ekin_rep[r] = 0.5 * m * np.sum(self.v[s][dyn[s]] ** 2)

    def step(self, dt, T, gamma, seed, step, slab_disp=None):
        d = C.c_double
        T = np.ascontiguousarray(np.broadcast_to(np.asarray(T, dtype=np.float64), (self.R,)))
        seed = np.ascontiguousarray(np.broadcast_to(np.asarray(seed, dtype=np.uint64), (self.R,)))
        if slab_disp is None:
            slab_disp = np.zeros(self.R)
        slab_disp = np.ascontiguousarray(np.broadcast_to(np.asarray(slab_disp, dtype=np.float64), (self.R,)))
        rc = lib().orc_md_step(C.byref(self.params), d(self.r_cut), C.c_int64(self.n), _p(self.x, d),
                               _p(self.v, d), _p(self.f, d), _p(self.flags, C.c_int32),
                               _p(self.zref, d), C.c_int32(self.R), _p(self.offsets, C.c_int32),
                               _p(self.lo, C.c_float), _p(self.hi, C.c_float), _p(self.per, C.c_uint8),
                               C.c_int(self.fp32_pred), d(dt), _p(T, d), d(gamma),
                               _p(seed, C.c_uint64), C.c_uint64(step), _p(slab_disp, d),
                               C.c_int(self.cells), _p(self.rho, d), _p(self.e_atom, d),
                               _p(self.e_rep, d), _p(self.w_rep, d), _p(self.ekin_rep, d))
        if rc != 0:
            raise RuntimeError(f"oracle md_step failed rc={rc}")
