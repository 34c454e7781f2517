"""Cell-centred grid fields (vx,vy,vz,bx,by,bz,rho), each [nz,ny,nx] float64, i fastest.

Random draws come from numpy PCG64 (host, device independent); the sum over Fourier
modes is evaluated with torch on `device` (plumbing: the bytes produced are handed
unchanged to both the oracle and the CUDA path).
"""
import math

import numpy as np
import torch

from .configs import LPWorkload


def _centres(w: LPWorkload, device):
    """Cell-centre coordinates per axis, and the same as a fraction of the box."""
    n = w.n
    out = []
    for d in range(3):
        lo, hi = w.xlo[d], w.xhi[d]
        i = torch.arange(n, dtype=torch.float64, device=device)
        out.append(lo + (i + 0.5) * ((hi - lo) / n))
    return out


def _draw_modes(rng, nmodes, kmax, vector):
    """Integer wave vectors with 1 <= |k| <= kmax (rejection from [-kmax,kmax]^3),
    phases, and amplitudes: |A| = 1/|k|; vector modes have A perpendicular to k."""
    ks = []
    while len(ks) < nmodes:
        k = rng.integers(-kmax, kmax + 1, size=3)
        k2 = int(k[0] ** 2 + k[1] ** 2 + k[2] ** 2)
        if 1 <= k2 <= kmax * kmax:
            ks.append(k)
    ks = np.array(ks, dtype=np.int64)
    phi = rng.uniform(0.0, 2.0 * math.pi, size=nmodes)
    kn = np.sqrt((ks ** 2).sum(axis=1))
    if not vector:
        return ks, phi, (1.0 / kn)[:, None]
    A = np.empty((nmodes, 3))
    for m in range(nmodes):
        while True:
            r = rng.normal(size=3)
            a = r - ks[m] * (r @ ks[m]) / (kn[m] ** 2)      # remove the component along k
            na = np.linalg.norm(a)
            if na > 1e-3:
                break
        A[m] = a / na / kn[m]
    return ks, phi, A


def _mode_sum(w: LPWorkload, ks, phi, A, device):
    """sum_m A_m cos(2 pi k_m . xi + phi_m) at the cell centres, xi in [0,1)^3."""
    n = w.n
    xi = (torch.arange(n, dtype=torch.float64, device=device) + 0.5) / n
    ncomp = A.shape[1]
    out = [torch.zeros((n, n, n), dtype=torch.float64, device=device) for _ in range(ncomp)]
    two_pi = 2.0 * math.pi
    for m in range(ks.shape[0]):
        px = (two_pi * float(ks[m, 0])) * xi
        py = (two_pi * float(ks[m, 1])) * xi
        pz = (two_pi * float(ks[m, 2])) * xi + float(phi[m])
        c = torch.cos(pz[:, None, None] + py[None, :, None] + px[None, None, :])
        for comp in range(ncomp):
            out[comp].add_(c, alpha=float(A[m, comp]))
        del c
    return out


def make_fields(w: LPWorkload, t: float = 0.0, device="cpu"):
    """Seven tensors in the order vx,vy,vz,bx,by,bz,rho at time t (t matters only for
    the homologous workload, reading R18: v = alpha x/(1+alpha t), rho = (1+alpha t)^-3)."""
    n = w.n
    dev = torch.device(device)
    shape = (n, n, n)
    zeros = lambda: torch.zeros(shape, dtype=torch.float64, device=dev)
    if w.field_kind == "uniform_b":
        return [zeros(), zeros(), zeros(), zeros(), zeros(),
                torch.full(shape, w.b0, dtype=torch.float64, device=dev),
                torch.ones(shape, dtype=torch.float64, device=dev)]
    if w.field_kind == "homologous":
        cx, cy, cz = _centres(w, dev)
        s = w.alpha / (1.0 + w.alpha * t)
        vx = (s * cx)[None, None, :].expand(shape).contiguous()
        vy = (s * cy)[None, :, None].expand(shape).contiguous()
        vz = (s * cz)[:, None, None].expand(shape).contiguous()
        rho = torch.full(shape, (1.0 + w.alpha * t) ** -3, dtype=torch.float64, device=dev)
        return [vx, vy, vz, zeros(), zeros(), zeros(), rho]
    if w.field_kind == "turbulent":
        rng = np.random.Generator(np.random.PCG64(w.seed))
        kv, pv, Av = _draw_modes(rng, w.nmodes, w.kmax, vector=True)
        kb, pb, Ab = _draw_modes(rng, w.nmodes, w.kmax, vector=True)
        kr, pr, Ar = _draw_modes(rng, w.nmodes, w.kmax, vector=False)
        v = _mode_sum(w, kv, pv, Av, dev)
        vmag = torch.sqrt(v[0] ** 2 + v[1] ** 2 + v[2] ** 2).max()
        v = [c * (w.vmax / vmag) for c in v]
        b = _mode_sum(w, kb, pb, Ab, dev)
        brms = torch.sqrt((b[0] ** 2 + b[1] ** 2 + b[2] ** 2).mean())
        b = [c * (w.brms / brms) for c in b]
        g = _mode_sum(w, kr, pr, Ar, dev)[0]
        g = g - g.mean()
        g = g / torch.sqrt((g ** 2).mean())
        rho = torch.exp(w.sigma_rho * g)
        return v + b + [rho]
    raise ValueError(w.field_kind)


def mean_magnetic_energy(fields7) -> float:
    """<|B|^2/2> over grid cells (for u_rad = frac * this, reading R6)."""
    bx, by, bz = fields7[3], fields7[4], fields7[5]
    return float((0.5 * (bx ** 2 + by ** 2 + bz ** 2)).mean())
