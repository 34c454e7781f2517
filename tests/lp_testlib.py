"""Shared helpers of the GPU parity tests: set up the oracle side and the CUDA side from the
same seeded inputs (lp_inputs) and compare them under the rules of DESIGN.md section 7."""
import numpy as np

import lp_inputs as I
from oracle import lp_oracle as orc

REL_TOL = 1e-10          # north_star: relative 1e-10 (fp64) for positions and spectra
CHI_FLOOR = 1e-290


def oracle_params(w, u_rad):
    return orc.make_params(w.n, w.n, w.n, w.xlo, w.xhi, w.periodic, w.nbins, w.e_min, w.e_max,
                           kappa=w.kappa, u_rad=u_rad, cfl_e=w.cfl_e, max_substeps=w.max_substeps)


def u_rad_of(w, fields):
    return w.u_rad_frac * I.mean_magnetic_energy(fields) if w.u_rad_frac > 0 else 0.0


def fields_to_numpy(fields):
    return [f.detach().cpu().numpy() for f in fields]


def workload1_dt(w):
    """dt = 0.9 C_E / lambda_top (reading R13): one substep per step for every particle."""
    E = I.bin_edges(w.nbins, w.e_min, w.e_max)
    cr = w.kappa * 0.5 * w.b0 ** 2
    lam_top = cr * E[-2] ** 2 / (E[-1] - E[-2])
    return 0.9 * w.cfl_e / lam_top


def assert_chi_close(got, want, tol=REL_TOL, what="chi"):
    got = np.asarray(got); want = np.asarray(want)
    assert got.shape == want.shape
    err = np.abs(got - want) / np.maximum(np.abs(want), CHI_FLOOR)
    bad = err > tol
    assert not bad.any(), "%s: %d of %d entries off, worst rel %.3e at %s" % (
        what, int(bad.sum()), bad.size, float(err.max()), np.unravel_index(int(err.argmax()), err.shape))


def assert_nsub_equal(got, want, note=""):
    got = np.asarray(got); want = np.asarray(want)
    bad = np.nonzero(got != want)[0]
    assert bad.size == 0, "n_sub differs for %d particles %s: first %s gpu=%s oracle=%s" % (
        bad.size, note, bad[:5], got[bad[:5]], want[bad[:5]])


def oracle_sort_state(prm, x, y, z, pid, chi):
    key = orc.cell_key(prm, x, y, z)
    perm = orc.sort_perm(key, pid)
    return x[perm], y[perm], z[perm], pid[perm], chi[perm], key[perm], perm
