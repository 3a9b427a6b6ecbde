"""Helpers shared by the GPU parity tests (tests only)."""
import numpy as np

from paper_2409_10383_b200 import inputs as I


def perturbation_scale(u, p):
    """S of DESIGN.md 'Tolerance': max over fields of |f - f_Minkowski|."""
    return float(np.abs(u - I.minkowski(p)).max())


def rel_err(a, b, floor):
    """per-field max|a-b| / max(max|b|, floor)"""
    out = np.zeros(a.shape[0])
    for f in range(a.shape[0]):
        scale = max(float(np.abs(b[f]).max()), floor)
        out[f] = float(np.abs(a[f] - b[f]).max()) / scale if scale > 0 else 0.0
    return out


def padded_reference(u, p):
    """State-with-ghosts [F][N_b][m][m][m] by the definition of O2: numpy's own wrap / edge padding of the
    global array, cut into blocks."""
    g = p.ng
    mode = "wrap" if p.bc == 0 else "edge"
    up = np.pad(u, ((0, 0), (g, g), (g, g), (g, g)), mode=mode)
    n, m = p.n, p.n + 2 * g
    out = np.empty((u.shape[0], p.nblocks, m, m, m))
    for bz in range(p.nb[2]):
        for by in range(p.nb[1]):
            for bx in range(p.nb[0]):
                b = (bz * p.nb[1] + by) * p.nb[0] + bx
                out[:, b] = up[:, bz * n:bz * n + m, by * n:by * n + m, bx * n:bx * n + m]
    return out
