"""Pins for the oracle's spectral update (coefficients, CFL substeps, donor-cell upwind).

What fixes the expected values: hand-worked tiny cases (tests/golden/spectral_handworked.txt),
the analytic solution of Eq. 6 along characteristics for pure synchrotron
losses (Eq. 4) and for adiabatic expansion, a scale-invariance identity of
the log grid, the discrete steady state, number conservation and positivity.
"""
import math

import numpy as np
import pytest

from oracle import lp_oracle as orc


def log_bins(nb, e_min, e_max):
    return orc.bin_table(nb, e_min, e_max)


# ------------------------------------------------------------------ hand-worked cases

@pytest.mark.parametrize("case", ["A", "B", "C", "D"])
def test_handworked_cases(golden, case):
    g = golden("spectral_handworked.txt")
    E = np.array(g[case + "_edges"]); dE = np.diff(E)
    a, cr, dtau = g[case + "_a_cr_dtau"]
    lam_e, nsub_e, lost_e = g[case + "_lambda_nsub_lost"]
    nsub, lam = orc.cfl_nsub(E, dE, a, cr, dtau, cfl_e=0.5)
    assert lam == lam_e and nsub == int(nsub_e)
    chi, lost = orc.spectral_row(E, dE, a, cr, dtau, nsub, g[case + "_chi_in"])
    assert np.max(np.abs(chi - np.array(g[case + "_chi_out"]))) < 1e-15
    assert abs(lost - lost_e) < 1e-15


def test_bin_table_geometry():
    E, dE, Ec = log_bins(64, 1e1, 1e6)
    assert E[0] == 1e1 and abs(E[-1] - 1e6) < 1e-9
    r = E[1:] / E[:-1]
    assert np.max(np.abs(r - 10 ** (5 / 64))) < 1e-14
    assert np.max(np.abs(dE - (E[1:] - E[:-1]))) == 0.0
    assert np.max(np.abs(Ec ** 2 / (E[1:] * E[:-1]) - 1)) < 1e-15


# ------------------------------------------------------------------ invariants

def test_no_forcing_leaves_row_bitwise_unchanged():
    E, dE, _ = log_bins(32, 1.0, 1e7)
    chi0 = np.random.default_rng(0).uniform(0.1, 2.0, 32)
    nsub, lam = orc.cfl_nsub(E, dE, 0.0, 0.0, 0.3)
    assert nsub == 1 and lam == 0.0
    chi, lost = orc.spectral_row(E, dE, 0.0, 0.0, 0.3, 1, chi0)
    assert np.array_equal(chi, chi0) and lost == 0.0


@pytest.mark.parametrize("seed", range(6))
def test_number_conservation_and_positivity(seed):
    """sum chi_i dE_i + lost is constant; chi stays >= 0 for C_E <= 1, also with a sign change."""
    rng = np.random.default_rng(100 + seed)
    nb = int(rng.choice([16, 64, 128]))
    E, dE, _ = log_bins(nb, 1.0, 1e6)
    chi0 = rng.uniform(0.0, 1.0, nb) * E[:-1] ** -2.0
    chi0[rng.integers(0, nb, 4)] = 0.0
    a = float(rng.normal()) * 3.0                 # both signs
    cr = float(10 ** rng.uniform(-8, -4))
    dtau = float(10 ** rng.uniform(-2, 0.5))
    nsub, lam = orc.cfl_nsub(E, dE, a, cr, dtau, cfl_e=0.5, max_substeps=1 << 30)
    assert nsub >= 1 and dtau * lam / nsub <= 0.5 * (1 + 1e-12)
    assert nsub == 1 or dtau * lam / (nsub - 1) > 0.5
    chi, lost = orc.spectral_row(E, dE, a, cr, dtau, nsub, chi0)
    n0 = orc.row_number(dE, chi0); n1 = orc.row_number(dE, chi)
    assert abs(n1 + lost - n0) < 1e-13 * n0
    assert (chi >= 0.0).all()


def test_cfl_lambda_brute_force_and_cap():
    E, dE, _ = log_bins(16, 1.0, 1e4)
    a, cr, dtau = -0.7, 3e-3, 0.9
    w = [-float(e) * (a + cr * float(e)) for e in E]
    lam_bf = max((max(w[i + 1], 0.0) - min(w[i], 0.0)) / float(dE[i]) for i in range(16))
    nsub, lam = orc.cfl_nsub(E, dE, a, cr, dtau)
    assert lam == lam_bf and nsub == math.ceil(dtau * lam_bf / 0.5)
    capped, _ = orc.cfl_nsub(E, dE, a, cr, dtau, max_substeps=3)
    assert nsub > 3 and capped == -3


# ------------------------------------------------------------------ scheme-exact identities

@pytest.mark.parametrize("a,p", [(0.8, 2.2), (-0.8, 2.2), (0.3, 3.0)])
def test_scale_invariance_product_formula(a, p):
    """On a log grid with w = -a*eps a power law chi ~ Ec^-p stays a power law and every interior
    bin is multiplied per substep by 1 + dts*a*(r^(1-p) - 1)/(r - 1)   (a > 0, donor = bin above)
    or                             1 - dts*a*(r^p - r)/(r - 1)         (a < 0, donor = bin below)."""
    nb = 128
    E, dE, Ec = log_bins(nb, 1.0, 1e7)
    r = (1e7) ** (1.0 / nb)
    chi0 = Ec ** -p
    dtau, steps = 0.04, 50
    chi = chi0.copy(); fac = 1.0
    for _ in range(steps):
        nsub, _ = orc.cfl_nsub(E, dE, a, 0.0, dtau)
        chi, _ = orc.spectral_row(E, dE, a, 0.0, dtau, nsub, chi)
        dts = dtau / nsub
        g = 1 + dts * a * (r ** (1 - p) - 1) / (r - 1) if a > 0 else 1 - dts * a * (r ** p - r) / (r - 1)
        fac *= g ** nsub
    ratio = chi / chi0
    interior = slice(60, 68)        # far from both ends: boundary effects travel <= 1 bin / substep
    assert np.max(np.abs(ratio[interior] / fac - 1)) < 1e-12
    assert (fac < 1) == (a > 0)     # expansion lowers chi at fixed eps (p > 1)


def test_pure_loss_steady_state_is_a_fixed_point():
    """chi_i = C/|w(E_i)| makes the donor-cell flux w_k chi_k uniform: interior bins do not move."""
    nb = 64
    E, dE, _ = log_bins(nb, 1e1, 1e6)
    cr = 5e-9
    chi0 = 1.0 / (cr * E[:-1] ** 2)
    dtau = 20.0
    nsub, _ = orc.cfl_nsub(E, dE, 0.0, cr, dtau)
    chi, _ = orc.spectral_row(E, dE, 0.0, cr, dtau, nsub, chi0)
    assert np.max(np.abs(chi[:nb - 1 - nsub] / chi0[:nb - 1 - nsub] - 1)) < 1e-13
    assert chi[-1] < chi0[-1]       # top bin drains: nothing flows in from above


# ------------------------------------------------------------------ analytic: synchrotron cooling

def cooled_bin_numbers(E, K, p, ea, eb, cr, t):
    """Exact bin contents of the cooled power law: number is conserved along the characteristics
    eps(t) = eps0/(1 + c_r eps0 t)  (solution of Eq. 4), so n_i = N0(eps0(E_{i+1})) - N0(eps0(E_i))."""
    def cum0(e0):
        e0 = np.clip(e0, ea, eb)
        return K * (e0 ** (1 - p) - ea ** (1 - p)) / (1 - p)
    with np.errstate(divide="ignore", invalid="ignore"):
        e0 = np.where(cr * E * t < 1.0, E / (1.0 - cr * E * t), np.inf)
    c = cum0(e0)
    return c[1:] - c[:-1]


def run_synchrotron(nb, full_path):
    """Workload 1 of BASELINE.json: B = (0,0,1e-4), v = 0, rho = 1, N_b bins on [1e1,1e6], power law
    p = 2.5 on [1e2,1e5], 100 steps with dt = 0.9*C_E/lambda_top (n_sub = 1; reading R13)."""
    e_min, e_max, ea, eb, p = 1e1, 1e6, 1e2, 1e5, 2.5
    E, dE, Ec = log_bins(nb, e_min, e_max)
    cr = 1.0 * 0.5 * (1e-4) ** 2
    lam_top = cr * E[nb - 1] ** 2 / dE[nb - 1]
    dt = 0.9 * 0.5 / lam_top
    steps = int(round(1.06 / (cr * eb) / dt))
    K = (1 - p) / (eb ** (1 - p) - ea ** (1 - p))
    chi = np.where((Ec >= ea) & (Ec <= eb), K * Ec ** -p, 0.0)
    n_init = float(np.sum(chi * dE))
    if full_path:
        n = 4
        prm = orc.make_params(n, n, n, (-1,) * 3, (1,) * 3, (1, 1, 1), nb, e_min, e_max, kappa=1.0)
        z = np.zeros((n, n, n))
        fields = [z, z, z, z, z, z + 1e-4, z + 1.0]
        rows = np.tile(chi, (3, 1))
        pos = np.array([-0.3, 0.1, 0.7])
        for _ in range(steps):
            rows, nsub, lost = orc.spectral_update(prm, fields, pos, pos, pos, np.ones(3), dt, rows)
            assert (nsub == 1).all()
        assert np.allclose(rows[0], rows[1], rtol=1e-11, atol=0.0)
        chi = rows[0]
    else:
        for _ in range(steps):
            nsub, _ = orc.cfl_nsub(E, dE, 0.0, cr, dt)
            assert nsub == 1
            chi, _ = orc.spectral_row(E, dE, 0.0, cr, dt, nsub, chi)
    t = steps * dt
    exact = cooled_bin_numbers(E, K, p, ea, eb, cr, t)
    cutoff = eb / (1 + cr * eb * t)
    smooth = (E[:-1] > 2e2) & (E[1:] < 0.5 * cutoff)
    err = np.max(np.abs(chi[smooth] * dE[smooth] / exact[smooth] - 1))
    l1 = np.sum(np.abs(chi * dE - exact)) / np.sum(exact)
    return err, l1, chi, dE, n_init


def test_synchrotron_cooled_power_law_first_order_convergence():
    errs = {nb: run_synchrotron(nb, full_path=False)[:2] for nb in (64, 128, 256)}
    assert errs[64][0] < 0.04 and errs[128][0] < 0.025 and errs[256][0] < 0.0125, errs
    assert errs[256][0] < 0.62 * errs[128][0] < 0.62 * 0.9 * errs[64][0] / 0.62, errs
    assert errs[64][1] < 0.08 and errs[256][1] < errs[128][1] < errs[64][1], errs


def test_synchrotron_through_the_full_update_path():
    """Same run through gather + coefficients: pins c_r = kappa |B|^2/2 and dtau = dt for v = 0."""
    err_row, l1_row, chi_row, dE, n_init = run_synchrotron(64, full_path=False)
    err, l1, chi, _, _ = run_synchrotron(64, full_path=True)
    assert np.max(np.abs(chi - chi_row)) <= 1e-12 * np.max(chi_row)
    assert err < 0.04
    # number conserved: nothing has reached the bottom edge yet
    assert abs(np.sum(chi * dE) - n_init) < 1e-12 * n_init
    assert 0.9 < n_init < 1.0       # point values at bin centres, support cuts through two bins


# ------------------------------------------------------------------ analytic: adiabatic + coefficients

@pytest.mark.parametrize("nb,tol", [(128, 0.12), (512, 0.035)])
def test_adiabatic_expansion_density_law(nb, tol):
    """Pure adiabatic change: eps ~ rho^{1/3}, so a power law's amplitude at fixed eps scales as
    (rho/rho0)^{(p-1)/3}.  Run through the full path: rho_old -> rho_new over 200 steps."""
    p = 2.2; n = 4; steps = 200; alpha = 0.1; dt = 0.04
    prm = orc.make_params(n, n, n, (-1,) * 3, (1,) * 3, (0, 0, 0), nb, 1.0, 1e7)
    E, dE, Ec = log_bins(nb, 1.0, 1e7)
    chi = (Ec ** -p)[None, :].copy()
    z = np.zeros((n, n, n)); pos = np.array([0.2])
    rho = lambda t: (1 + alpha * t) ** -3
    for s in range(steps):
        fields = [z, z, z, z, z, z, z + rho((s + 1) * dt)]
        chi, nsub, lost = orc.spectral_update(prm, fields, pos, pos, pos, np.array([rho(s * dt)]), dt, chi)
    ratio = chi[0] / Ec ** -p
    expect = rho(steps * dt) ** ((p - 1) / 3)
    mid = slice(nb // 4, nb // 2)
    assert expect < 1
    assert np.max(np.abs(ratio[mid] / expect - 1)) < tol
    assert ratio[mid].mean() < 1 and ratio[mid].mean() > expect * (1 - 1e-3)   # diffusion errs high


def test_coefficients_closed_values():
    prm = orc.make_params(4, 4, 4, (-1,) * 3, (1,) * 3, (1, 1, 1), 8, 1.0, 1e4, kappa=2.0, u_rad=0.25)
    a, cr, dtau = orc.coefficients(prm, 0.5, (0.6, 0.0, 0.0), (0.0, 3.0, 4.0), 2.0, 1.0)
    assert abs(dtau - 0.5 * 0.8) < 1e-16                        # gamma_g = 1.25
    assert abs(cr - 2.0 * (12.5 + 0.25)) < 1e-14                # kappa (|B|^2/2 + u_rad)
    assert abs(a - (-math.log(2.0) / (3 * 0.4))) < 1e-15        # compression => a < 0
    a2, _, _ = orc.coefficients(prm, 0.5, (0, 0, 0), (0, 0, 0), 0.5, 1.0)
    assert a2 > 0                                               # expansion => a > 0 => energy loss


def test_moving_fluid_cools_slower_by_gamma():
    """dtau = dt/gamma_g: with |v| = 0.6 a step of dt equals a rest-frame step of 0.8 dt."""
    nb = 64; n = 4
    prm = orc.make_params(n, n, n, (-1,) * 3, (1,) * 3, (1, 1, 1), nb, 1e1, 1e6)
    E, dE, Ec = log_bins(nb, 1e1, 1e6)
    z = np.zeros((n, n, n)); pos = np.array([0.0]); chi0 = (Ec ** -2.5)[None, :]
    mov, _, _ = orc.spectral_update(prm, [z + 0.6, z, z, z, z, z + 1e-4, z + 1], pos, pos, pos, np.ones(1), 10.0, chi0)
    rest, _, _ = orc.spectral_update(prm, [z, z, z, z, z, z + 1e-4, z + 1], pos, pos, pos, np.ones(1), 8.0, chi0)
    assert np.max(np.abs(mov / rest - 1)) < 1e-13
