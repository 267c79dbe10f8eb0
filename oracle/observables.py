"""Observables of the paper's tensile tests, fp64 numpy: virial stress and engineering strain.

TEST INFRASTRUCTURE ONLY, like the rest of oracle/: imported by tests/ alone; shares nothing with the CUDA path.

Eq.5 is garbled in the source (reading A11); the standard virial stress it stands for is
    sigma_ab = -(1/V) [ W_ab + K_ab ],   W_ab = 1/2 sum_i sum_j d_ij,a f_ij,b,   K_ab = sum_i m v_i,a v_i,b,
tension positive, with V "calculated from the hard-sphere volumes" and held constant: V is an input here.
W_ab is what oracle.compute returns as w_rep; K runs over the dynamic atoms (grips are rigid, D:A12).
Eq.4: strain = (L - L0) / L0.
"""
import numpy as np

ACC = 9.648533212e-3          # 1 eV/(A amu) in A/fs^2: (m/ACC) v^2 is an energy in eV for m in amu, v in A/fs
EV_PER_A3_IN_GPA = 160.21766208


def kinetic_tensor(v, flags, offsets, mass_amu):
    """K_ab of every replica, order xx yy zz xy xz yz, eV.  v: (n,3) A/fs; flags: (n,) 0 = dynamic."""
    v = np.asarray(v, dtype=np.float64)
    R = len(offsets) - 1
    out = np.zeros((R, 6))
    m = mass_amu / ACC
    for r in range(R):
        s = slice(offsets[r], offsets[r + 1])
        vv = v[s][np.asarray(flags[s]) == 0]
        out[r] = m * np.array([np.sum(vv[:, 0] * vv[:, 0]), np.sum(vv[:, 1] * vv[:, 1]), np.sum(vv[:, 2] * vv[:, 2]),
                               np.sum(vv[:, 0] * vv[:, 1]), np.sum(vv[:, 0] * vv[:, 2]), np.sum(vv[:, 1] * vv[:, 2])])
    return out


def stress(w_rep, k_rep, volume):
    """sigma_ab = -(W_ab + K_ab) / V per replica (eV/A^3, tension positive); multiply by EV_PER_A3_IN_GPA for GPa."""
    w_rep, k_rep = np.asarray(w_rep, dtype=np.float64), np.asarray(k_rep, dtype=np.float64)
    return -(w_rep + k_rep) / np.asarray(volume, dtype=np.float64)[:, None]


def strain(length, length0):
    """Eq.4."""
    return (np.asarray(length, dtype=np.float64) - length0) / length0
