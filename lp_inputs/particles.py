"""Particle positions, ids and initial spectra (numpy, PCG64-seeded)."""
import numpy as np

from .configs import LPWorkload


def bin_edges(nbins, e_min, e_max):
    """Log-spaced edges used ONLY to place the initial spectrum (input data); the oracle
    and the CUDA library each build their own bin table."""
    k = np.arange(nbins + 1, dtype=np.float64)
    return e_min * (e_max / e_min) ** (k / nbins)


def make_particles(w: LPWorkload, shuffle_ids: bool = False):
    """x, y, z uniform in pos_box^3 (float64) and unique ids (uint64)."""
    rng = np.random.Generator(np.random.PCG64(w.seed + 1000))
    lo, hi = w.pos_box
    x = rng.uniform(lo, hi, size=w.np)
    y = rng.uniform(lo, hi, size=w.np)
    z = rng.uniform(lo, hi, size=w.np)
    pid = np.arange(w.np, dtype=np.uint64)
    if shuffle_ids:
        pid = rng.permutation(pid)
    return x, y, z, pid


def make_spectrum(w: LPWorkload, jitter: bool = True, n0: float = 1.0):
    """chi[np, nbins]: Eq. 13 evaluated at the geometric bin centres,
    chi_i = N0 (1-p)/(eb^{1-p} - ea^{1-p}) Ec_i^{-p} on the support [ea, eb], zero outside.
    jitter multiplies row p by (1 + 0.5 u_p) so that a mis-permuted row shows up."""
    E = bin_edges(w.nbins, w.e_min, w.e_max)
    Ec = np.sqrt(E[:-1] * E[1:])
    ea, eb = w.support if w.support is not None else (w.e_min, w.e_max)
    p = w.p_index
    norm = n0 * (1.0 - p) / (eb ** (1.0 - p) - ea ** (1.0 - p))
    row = np.where((Ec >= ea) & (Ec <= eb), norm * Ec ** (-p), 0.0)
    chi = np.tile(row, (w.np, 1))
    if jitter:
        rng = np.random.Generator(np.random.PCG64(w.seed + 2000))
        chi *= (1.0 + 0.5 * rng.uniform(size=w.np))[:, None]
    return np.ascontiguousarray(chi)
