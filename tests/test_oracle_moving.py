"""Pins of the oracle's per-particle moving energy grid (NEXT-5; readings E1-E4 of DESIGN.md section 3).

What the paper and the mathematics fix: the characteristics of Eq. 6 have the closed forms
north_star quotes -- E0/(1 + c B^2 E0 t) for synchrotron losses, E ~ rho^(1/3) for adiabatic expansion -- and
Eq. 6 conserves the number between two characteristics.  Hand-worked values (tests/golden/
moving_grid_handworked.txt), an independent ODE integration for the combined case, exactness on a cooled power
law, the semigroup property, and the full path through gather and coefficients in homologous flow."""
import numpy as np
import pytest
from scipy.integrate import quad, solve_ivp

import lp_inputs as I
from oracle import lp_oracle as orc
from lp_testlib import fields_to_numpy, oracle_params

E5 = np.array([1.0, 10.0, 100.0, 1000.0, 10000.0])


def test_handworked(golden):
    g = golden("moving_grid_handworked.txt")
    eng, chi = orc.moving_row(0.0, 1e-4, 1.0, E5, np.ones(4))
    assert np.allclose(eng, g["A_eng"], rtol=1e-15, atol=0) and np.allclose(chi, g["A_chi"], rtol=2e-15, atol=0)
    s = g["B_s"][0]
    eng, chi = orc.moving_row(s / 2.0, 0.0, 2.0, E5, np.ones(4))            # a dtau = s
    assert np.allclose(eng, g["B_eng"], rtol=4e-16, atol=0) and np.allclose(chi, g["B_chi"], rtol=1e-15, atol=0)
    eng, chi = orc.moving_row(s, 1e-4, 1.0, E5, np.ones(4))
    assert np.isclose(eng[-1], g["C_top"][0], rtol=1e-11)
    assert np.isclose(eng[-1], 5000.0 / (1.0 + g["C_beta"][0] * 10000.0), rtol=1e-15)


@pytest.mark.parametrize("a,cr", [(0.3, 2e-3), (-0.4, 5e-4), (1e-9, 1e-3), (-2.0, 0.0), (0.0, 1e-2), (3.0, 1e-6)])
def test_edges_follow_the_ode_of_eq6(a, cr):
    """d(eps)/d(tau) = -eps (a + c_r eps), integrated numerically (independent of the closed form)."""
    dtau = 0.7
    E = np.logspace(0, 4, 9)
    eng, _ = orc.moving_row(a, cr, dtau, E, np.ones(8))
    sol = solve_ivp(lambda t, e: -e * (a + cr * e), (0.0, dtau), E, rtol=1e-12, atol=1e-14, method="DOP853")
    assert np.allclose(eng, sol.y[:, -1], rtol=2e-10, atol=0)


def test_synchrotron_law_after_many_steps():
    """north_star: E(t) = E0 / (1 + c B^2 E0 t), here c B^2 = c_r; 100 steps against the one-shot formula."""
    cr, dtau, n = 3e-6, 0.25, 100
    E, dE, Ec = orc.bin_table(64, 1e1, 1e6)
    eng, chi = E.copy(), np.ones(64)
    num0 = chi * dE
    for _ in range(n):
        eng, chi = orc.moving_row(0.0, cr, dtau, eng, chi)
    assert np.allclose(eng, E / (1.0 + cr * E * dtau * n), rtol=1e-13, atol=0)
    assert np.allclose(chi * np.diff(eng), num0, rtol=1e-12, atol=0)         # bin numbers unchanged (E3)


def test_semigroup_and_number_conservation_with_both_terms():
    rng = np.random.default_rng(2)
    E, dE, Ec = orc.bin_table(128, 1.0, 1e7)
    chi0 = rng.uniform(0.5, 1.5, size=128) * Ec ** -2.2
    a, cr, dtau = -0.35, 4e-7, 0.9
    e1, c1 = orc.moving_row(a, cr, dtau, E, chi0)
    e2, c2 = orc.moving_row(a, cr, dtau / 2, E, chi0)
    e2, c2 = orc.moving_row(a, cr, dtau / 2, e2, c2)
    assert np.allclose(e1, e2, rtol=1e-14, atol=0) and np.allclose(c1, c2, rtol=1e-12, atol=0)
    assert np.allclose(c1 * np.diff(e1), chi0 * dE, rtol=1e-12, atol=0)
    assert np.all(np.diff(e1) > 0)                                           # characteristics do not cross


def test_cooled_power_law_is_exact_in_bin_means():
    """chi0 = exact bin means of K eps^-p; pure synchrotron cooling.  The analytic solution
    N(eps, t) = K eps^-p (1 - c_r eps t)^(p-2) averaged over the moved bins must come out to rounding --
    unlike the fixed-grid donor-cell scheme, whose error is first order (tests/test_oracle_spectral.py)."""
    p, cr, t = 2.5, 2e-6, 1.0
    E, dE, Ec = orc.bin_table(32, 1e2, 1e5)
    chi = (E[:-1] ** (1 - p) - E[1:] ** (1 - p)) / ((p - 1) * dE)
    eng = E.copy()
    for _ in range(10):
        eng, chi = orc.moving_row(0.0, cr, t / 10, eng, chi)
    for i in (0, 7, 20, 31):
        want = quad(lambda e: e ** -p * (1 - cr * e * t) ** (p - 2), eng[i], eng[i + 1], epsabs=0, epsrel=1e-12)[0]
        assert np.isclose(chi[i] * (eng[i + 1] - eng[i]), want, rtol=1e-10)


def test_adiabatic_law_through_the_whole_path():
    """Homologous expansion (workload 2, reading R18), staged as the product does it: after every step the
    edges must have scaled by (rho(t)/rho_0)^(1/3) (north_star: E ~ rho^(1/3)), B = 0, v << 1."""
    w = I.workload(2).scaled(n=16, np=64, nbins=16)
    prm = oracle_params(w, 0.0)
    x, y, z, pid = I.make_particles(w)
    E, dE, Ec = orc.bin_table(w.nbins, w.e_min, w.e_max)
    eng = np.tile(E, (w.np, 1)); chi = np.ones((w.np, w.nbins))
    t = 0.0
    for k in range(20):
        f0 = fields_to_numpy(I.make_fields(w, t=t, device="cpu"))
        f1 = fields_to_numpy(I.make_fields(w, t=t + w.dt, device="cpu"))
        k1, rho_old, xs = orc.push_stage0(prm, f0, x, y, z, w.dt)
        x, y, z, status = orc.push_stage1(prm, f1, x, y, z, xs, k1, w.dt)
        eng, chi = orc.moving_update(prm, f1, x, y, z, rho_old, w.dt, eng, chi)
        t += w.dt
    rho_ratio = (1.0 + w.alpha * t) ** -3
    assert np.allclose(eng, E[None, :] * rho_ratio ** (1.0 / 3.0), rtol=1e-13, atol=0)
    assert np.allclose(chi * np.diff(eng, axis=1), dE[None, :], rtol=1e-12, atol=0)
