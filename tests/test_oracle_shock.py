"""Pins of the oracle's shock-crossing update (Eq. 7-8; readings S1-S4 of DESIGN.md).

What fixes it other than itself: two cases worked by hand in exact fractions (tests/golden/
shock_handworked.txt); the closed form of the integral for a power-law input; the post-shock slope
q - 2 the paper prints for its planar-shock test (r ~= 3.64, slope 2.14, 0.5 % error: PAPER.md:274-290);
number conservation, linearity, causality (nothing appears below the lowest occupied bin), and the
"no shock" case.
"""
import numpy as np
import pytest

from oracle import lp_oracle as orc


@pytest.mark.parametrize("case", ["A", "B"])
def test_shock_handworked(golden, case):
    g = golden("shock_handworked.txt")
    E = np.array(g[case + "_edges"]); dE = np.diff(E)
    r, q_r = g[case + "_r_qr"]
    out, changed = orc.shock_row(E, dE, r, q_r, g[case + "_chi_in"])
    assert changed
    assert np.max(np.abs(out - np.array(g[case + "_chi_out"]))) < 1e-15


def test_shock_slope_of_the_papers_planar_shock(golden):
    """Steep injected spectrum (Eq. 13 with the paper's p = 9, 128 bins on [1e2, 1e4]) through a shock of
    the paper's compression ratio: the post-shock spectrum is a power law of index q - 2."""
    g = golden("shock_arithmetic.txt")
    gam, rho_u, p_u, v_u = 5.0 / 3.0, 50.0, 0.01, 0.1
    M2 = v_u ** 2 / (gam * p_u / rho_u)
    r = (gam + 1) * M2 / (2 + (gam - 1) * M2)                 # Eq. 12
    assert abs(r - g["r"][0]) < 5e-3                          # "~= 3.64"
    q = 3 * r / (r - 1)                                       # Eq. 8, q_R = 0
    assert abs((q - 2) - g["slope"][0]) < 5e-3                # "q = 2.14" of Fig. 2
    E, dE, Ec = orc.bin_table(128, 1e2, 1e4)
    chi = Ec ** -9.0
    out, changed = orc.shock_row(E, dE, r, 0.0, chi)
    assert changed
    sel = (Ec > 3e2) & (Ec < 3e3)
    slope = -np.polyfit(np.log(Ec[sel]), np.log(out[sel]), 1)[0]
    assert abs(slope - (q - 2)) / (q - 2) < 5e-3              # the paper's own 0.5 %


@pytest.mark.parametrize("p", [1.2, 2.5])
def test_shock_closed_form_for_a_power_law(p):
    """chi_in = e^-p on the whole table: Int_{e_min}^{e} e'^(q-3-p) de' in closed form; the midpoint sum
    converges to it at second order in the bin ratio."""
    r, q = 4.0, 4.0
    errs = []
    for nb in (128, 512):
        E, dE, Ec = orc.bin_table(nb, 1.0, 1e4)
        out, _ = orc.shock_row(E, dE, r, 0.0, Ec ** -p)
        s = q - 2 - p
        exact = Ec ** (2 - q) * (Ec ** s - E[0] ** s) / s
        exact *= (Ec ** -p * dE).sum() / (exact * dE).sum()          # same normalisation
        sel = Ec > 10.0
        errs.append(np.max(np.abs(out[sel] / exact[sel] - 1)))
    assert errs[0] < 2e-2 and errs[1] < errs[0] / 8


def test_shock_conserves_number_and_is_linear_and_causal():
    rng = np.random.default_rng(5)
    E, dE, Ec = orc.bin_table(64, 1.0, 1e8)
    chi = rng.uniform(0.0, 1.0, 64) * Ec ** -2.0
    chi[:10] = 0.0
    out, changed = orc.shock_row(E, dE, 3.2, 0.1, chi)
    assert changed and (out >= 0).all()
    assert abs((out * dE).sum() / (chi * dE).sum() - 1) < 1e-14
    assert (out[:10] == 0.0).all() and out[10] > 0                   # nothing below the lowest occupied bin
    out3, _ = orc.shock_row(E, dE, 3.2, 0.1, 3.0 * chi)
    pos = out > 0
    assert np.max(np.abs(out3[pos] / (3.0 * out[pos]) - 1)) < 1e-14          # (3x is not exact in fp)


def test_no_shock_and_empty_rows_are_untouched():
    E, dE, Ec = orc.bin_table(32, 1.0, 1e4)
    chi = Ec ** -2.2
    for r in (1.0, 0.0, -3.0, float("nan")):
        out, changed = orc.shock_row(E, dE, r, 0.0, chi)
        assert not changed and np.array_equal(out, chi)
    out, changed = orc.shock_row(E, dE, 4.0, 0.0, np.zeros(32))
    assert not changed and (out == 0).all()


def test_shock_update_applies_row_by_row():
    rng = np.random.default_rng(11)
    E, dE, Ec = orc.bin_table(16, 1.0, 1e8)
    chi = rng.uniform(0.5, 1.5, (7, 16)) * Ec ** -2.5
    r = np.array([1.0, 2.0, 3.9, 0.5, 4.0, 1.0, 3.0])
    out = orc.shock_update(E, dE, r, 0.0, chi)
    for p in range(7):
        row, _ = orc.shock_row(E, dE, r[p], 0.0, chi[p])
        assert np.array_equal(out[p], row)


def test_shock_on_per_particle_grids_is_the_row_update_on_each_grid():
    """orc_shock_update_grid: every row on its own edges.  A particle whose grid is the fixed table must give
    orc_shock_update's row; a grid scaled by a factor s gives the same chi / s on the scaled bins (Eq. 7 is
    homogeneous in the energy: the update commutes with a rescaling of the energy axis); number is conserved."""
    nb = 32
    E, dE, Ec = orc.bin_table(nb, 1.0, 1e6)
    rng = np.random.default_rng(4)
    chi = rng.uniform(0.5, 1.5, size=(3, nb)) * Ec[None, :] ** -2.3
    s = 0.37
    eng = np.stack([E, s * E, E])
    chi_in = chi.copy(); chi_in[1] = chi[0] / s           # the same particle as row 0 on a scaled energy axis
    r = np.array([3.0, 3.0, 1.0])
    out = orc.shock_update_grid(eng, r, 0.1, chi_in)
    want0 = orc.shock_update(E, dE, r[:1], 0.1, chi[:1])[0]
    assert np.allclose(out[0], want0, rtol=1e-14, atol=0)
    assert np.allclose(out[1] * s, out[0], rtol=1e-12, atol=0)
    assert np.array_equal(out[2], chi_in[2])                # r = 1: untouched
    for p in range(2):
        w = np.diff(eng[p])
        assert np.isclose((out[p] * w).sum(), (chi_in[p] * w).sum(), rtol=1e-13)
