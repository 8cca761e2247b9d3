"""Brute-force restatement of PAPER.md Eq.(1) in numpy, used ONLY by the tests as an
independent pin for the oracle (no oracle code, no tables, no local energies)."""
import numpy as np


def distance_matrix(L):
    """r_ij: Euclidean minimum-image distance on the L x L torus."""
    s = np.arange(L * L)
    y, x = s // L, s % L
    dy = np.abs(y[:, None] - y[None, :]); dy = np.minimum(dy, L - dy)
    dx = np.abs(x[:, None] - x[None, :]); dx = np.minimum(dx, L - dx)
    return np.sqrt((dy * dy + dx * dx).astype(float))


def hamiltonian(n, phi, L, nu=0.5):
    """H = sum phi_i n_i + 1/2 sum_{i != j} (n_i - nu)(n_j - nu)/r_ij   (Eq.(1), E = 0)."""
    r = distance_matrix(L)
    with np.errstate(divide="ignore"):
        v = np.where(r > 0, 1.0 / r, 0.0)
    q = np.asarray(n, float) - nu
    return float(np.dot(phi, n) + 0.5 * q @ v @ q)


def min_image(d, L):
    d = d % L
    return d - L if d > L // 2 else d
