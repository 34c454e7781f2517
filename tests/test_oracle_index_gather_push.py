"""Pins for the oracle's cell key, sort, trilinear gather and two-stage pusher.

None of these re-types the oracle's formulas: each compares with something the paper
or the mathematics fixes (brute force, exactness properties, the closed form Eq. 10).
"""
import math

import numpy as np
import pytest

from oracle import lp_oracle as orc


def params(n=(8, 8, 8), periodic=(1, 1, 1), xlo=(-1, -1, -1), xhi=(1, 1, 1), nbins=8):
    return orc.make_params(n[0], n[1], n[2], xlo, xhi, periodic, nbins, 1.0, 1e4)


def grid_coords(prm):
    cs = []
    for d, n in enumerate((prm.nx, prm.ny, prm.nz)):
        lo, hi = prm.xlo[d], prm.xhi[d]
        cs.append(lo + (np.arange(n) + 0.5) * (hi - lo) / n)
    Z, Y, X = np.meshgrid(cs[2], cs[1], cs[0], indexing="ij")
    return X, Y, Z


# ------------------------------------------------------------------ key / sort

def test_cell_key_brute_force():
    """key == the cell whose faces bracket the particle (search over faces)."""
    rng = np.random.default_rng(1)
    prm = params(n=(5, 7, 3), xlo=(-1, 0, 2), xhi=(1, 3.5, 2.75))
    npart = 64
    x = rng.uniform(-1, 1, npart); y = rng.uniform(0, 3.5, npart); z = rng.uniform(2, 2.75, npart)
    # a few particles exactly on faces: a face belongs to the upper cell
    x[0] = -1.0; x[1] = -1 + 2 * 2 / 5; y[2] = 0.5 * 3; z[3] = 2.0
    key = orc.cell_key(prm, x, y, z)
    for p in range(npart):
        c = []
        for d, (v, n) in enumerate(((x[p], 5), (y[p], 7), (z[p], 3))):
            faces = prm.xlo[d] + np.arange(n + 1) * (prm.xhi[d] - prm.xlo[d]) / n
            found = [i for i in range(n) if faces[i] <= v < faces[i + 1]]
            assert len(found) == 1
            c.append(found[0])
        assert key[p] == (c[2] * 7 + c[1]) * 5 + c[0]


def test_cell_key_clamps_outside():
    prm = params(n=(4, 4, 4))
    key = orc.cell_key(prm, [-1.5, 1.0, 2.0], [0.0, 0.0, 0.0], [0.0, 0.0, 0.0])
    base = (2 * 4 + 2) * 4
    assert list(key) == [base + 0, base + 3, base + 3]


def test_sort_perm_selection_sort():
    rng = np.random.default_rng(2)
    n = 200
    key = rng.integers(0, 12, n).astype(np.uint32)      # many ties
    pid = rng.permutation(n).astype(np.uint64) + 7
    perm = orc.sort_perm(key, pid)
    # O(N^2) selection of the minimum (key, id) among the remaining
    remaining = list(range(n)); expect = []
    while remaining:
        best = remaining[0]
        for r in remaining[1:]:
            if (key[r], pid[r]) < (key[best], pid[best]):
                best = r
        expect.append(best); remaining.remove(best)
    assert list(perm) == expect
    assert sorted(perm) == list(range(n))


# ------------------------------------------------------------------ gather

def test_gather_constant_field_partition_of_unity():
    rng = np.random.default_rng(3)
    prm = params(n=(6, 5, 4))
    consts = [1.5, -2.0, 3.25, 1e-4, -7.0, 0.125, 42.0]
    fields = [np.full((4, 5, 6), c) for c in consts]
    x, y, z = (rng.uniform(-1, 1, 500) for _ in range(3))
    out = orc.gather(prm, fields, x, y, z)
    for m, c in enumerate(consts):
        assert np.max(np.abs(out[m] - c)) <= 2e-15 * abs(c)


@pytest.mark.parametrize("periodic", [(1, 1, 1), (0, 0, 0)])
def test_gather_linear_field_exact_in_interior(periodic):
    """Trilinear interpolation reproduces any field linear in x, y, z between cell centres."""
    rng = np.random.default_rng(4)
    prm = params(n=(8, 6, 10), periodic=periodic)
    X, Y, Z = grid_coords(prm)
    coef = rng.normal(size=(7, 4))
    fields = [c[0] + c[1] * X + c[2] * Y + c[3] * Z for c in coef]
    # stay between the first and last cell centres on every axis (away from seam / clamp)
    x = rng.uniform(-1 + 1 / 8, 1 - 1 / 8, 400)
    y = rng.uniform(-1 + 1 / 6, 1 - 1 / 6, 400)
    z = rng.uniform(-1 + 1 / 10, 1 - 1 / 10, 400)
    out = orc.gather(prm, fields, x, y, z)
    for m, c in enumerate(coef):
        exact = c[0] + c[1] * x + c[2] * y + c[3] * z
        assert np.max(np.abs(out[m] - exact)) < 1e-14 * np.abs(coef).sum()


def test_gather_axes_not_transposed():
    """A field that depends on one axis only must vary along that axis only."""
    prm = params(n=(4, 6, 8))
    X, Y, Z = grid_coords(prm)
    zeros = np.zeros_like(X)
    out = orc.gather(prm, [X, Y, Z, zeros, zeros, zeros, zeros + 1],
                     [0.1, 0.3], [-0.2, -0.2], [0.4, 0.4])
    assert abs(out[0, 0] - 0.1) < 1e-15 and abs(out[0, 1] - 0.3) < 1e-15
    assert abs(out[1, 0] + 0.2) < 1e-15 and abs(out[2, 0] - 0.4) < 1e-15


def test_gather_at_cell_centres_returns_cell_values():
    rng = np.random.default_rng(5)
    prm = params(n=(4, 4, 4))
    fields = [rng.normal(size=(4, 4, 4)) for _ in range(7)]
    X, Y, Z = grid_coords(prm)
    out = orc.gather(prm, fields, X.ravel(), Y.ravel(), Z.ravel())
    for m in range(7):
        assert np.max(np.abs(out[m] - fields[m].ravel())) < 1e-15


def test_gather_periodic_seam_and_clamp():
    """x at the domain edge: periodic averages first and last cell; clamped returns the edge cell."""
    f = np.zeros((2, 2, 4)); f[:, :, 0] = 1.0; f[:, :, 3] = 3.0
    fields = [f] * 7
    per = orc.gather(params(n=(4, 2, 2), periodic=(1, 1, 1)), fields, [-1.0], [0.0], [0.0])
    clp = orc.gather(params(n=(4, 2, 2), periodic=(0, 1, 1)), fields, [-1.0], [0.0], [0.0])
    assert abs(per[0, 0] - 2.0) < 1e-15 and abs(clp[0, 0] - 1.0) < 1e-15


# ------------------------------------------------------------------ push

def uniform_fields(n, v, rho=1.0):
    shape = (n[2], n[1], n[0])
    return [np.full(shape, v[0]), np.full(shape, v[1]), np.full(shape, v[2]),
            np.zeros(shape), np.zeros(shape), np.zeros(shape), np.full(shape, rho)]


def test_push_uniform_velocity_is_exact():
    """Test A of the paper: uniform v = (0.2, 0.2, 0.2) => x = x0 + v t, wrapped."""
    prm = params(n=(8, 8, 8))
    fields = uniform_fields((8, 8, 8), (0.2, 0.2, 0.2))
    rng = np.random.default_rng(6)
    x, y, z = (rng.uniform(-1, 1, 100) for _ in range(3))
    x0, y0, z0 = x.copy(), y.copy(), z.copy()
    dt, nsteps = 0.05, 300          # t = 15: several box crossings
    for _ in range(nsteps):
        k1, rho_old, xs = orc.push_stage0(prm, fields, x, y, z, dt)
        x, y, z, st = orc.push_stage1(prm, fields, x, y, z, xs, k1, dt)
        assert not st.any()
    for a, a0 in ((x, x0), (y, y0), (z, z0)):
        exact = (a0 + 0.2 * dt * nsteps + 1.0) % 2.0 - 1.0
        d = np.abs(a - exact); d = np.minimum(d, 2.0 - d)
        assert d.max() < 1e-13
        assert (a >= -1.0).all() and (a < 1.0).all()


def eq10(t):
    s3 = math.sqrt(3.0)
    return 2.0 / math.pi * math.atan(0.5 * (s3 * math.tan(math.pi * (s3 + 9.0 * t) / (6.0 * s3)) - 1.0))


def test_eq10_golden_value(golden):
    g = golden("pusher_eq10.txt")
    assert abs(eq10(g["t"][0]) - g["x_mod2"][0]) < 1e-10


def advect_eq9(n, t_end, cfl=0.5):
    prm = params(n=(n, 2, 2))
    xc = -1 + (np.arange(n) + 0.5) * 2.0 / n
    vx = np.broadcast_to(2.0 + np.sin(math.pi * xc), (2, 2, n)).copy()
    zeros = np.zeros_like(vx)
    fields = [vx, zeros, zeros, zeros, zeros, zeros, zeros + 1]
    nsteps = int(math.ceil(t_end / (cfl * (2.0 / n) / 3.0)))
    dt = t_end / nsteps
    x = np.array([0.0]); y = np.array([0.1]); z = np.array([-0.3])
    for _ in range(nsteps):
        k1, _, xs = orc.push_stage0(prm, fields, x, y, z, dt)
        x, y, z, _ = orc.push_stage1(prm, fields, x, y, z, xs, k1, dt)
    assert y[0] == 0.1 and z[0] == -0.3
    return x[0]


def test_push_matches_eq10_second_order(golden):
    """Simple-advection benchmark of section 4.1.1: the error against the
    closed form Eq. 10 at t = 10 falls as n^-2 for the two-stage scheme."""
    g = golden("pusher_eq10.txt")
    exact = g["x_mod2"][0]
    errs = []
    for n in (32, 64, 128, 256):
        xn = advect_eq9(n, g["t"][0])
        d = abs(xn - exact); errs.append(min(d, 2.0 - d))
    assert errs[-1] < 2e-4
    slopes = [math.log2(errs[i] / errs[i + 1]) for i in range(3)]
    assert all(abs(s - g["order"][0]) < 0.25 for s in slopes), (errs, slopes)


def test_push_homologous_staged_fields_exact():
    """v = alpha x/(1 + alpha t) with the field advanced between the stages (reading R18):
    Heun is exact, x = x0 (1 + alpha t); rho_old is the density of the stage-0 field."""
    n = 16; alpha = 0.1; dt = 0.04
    prm = params(n=(n, n, n), periodic=(0, 0, 0))
    X, Y, Z = grid_coords(prm)

    def fields_at(t):
        s = alpha / (1 + alpha * t)
        zeros = np.zeros_like(X)
        return [s * X, s * Y, s * Z, zeros, zeros, zeros, zeros + (1 + alpha * t) ** -3]

    rng = np.random.default_rng(7)
    x, y, z = (rng.uniform(-0.5, 0.5, 50) for _ in range(3))
    x0 = x.copy()
    t = 0.0
    for _ in range(100):
        k1, rho_old, xs = orc.push_stage0(prm, fields_at(t), x, y, z, dt)
        assert np.allclose(rho_old, (1 + alpha * t) ** -3, rtol=1e-14)
        x, y, z, st = orc.push_stage1(prm, fields_at(t + dt), x, y, z, xs, k1, dt)
        t += dt
    assert np.max(np.abs(x - x0 * (1 + alpha * t))) < 1e-13
    assert not st.any()


def test_push_status_flags_outside_on_open_axis():
    prm = params(n=(4, 4, 4), periodic=(0, 1, 1))
    fields = uniform_fields((4, 4, 4), (0.5, 0.0, 0.0))
    x = np.array([0.9, 0.0]); y = np.zeros(2); z = np.zeros(2)
    k1, _, xs = orc.push_stage0(prm, fields, x, y, z, 0.4)
    x, y, z, st = orc.push_stage1(prm, fields, x, y, z, xs, k1, 0.4)
    assert list(st) == [1, 0] and abs(x[0] - 1.1) < 1e-15


def test_step_equals_stages_and_threads_do_not_change_bits():
    rng = np.random.default_rng(8)
    n = 8
    prm = orc.make_params(n, n, n, (-1,) * 3, (1,) * 3, (1, 1, 1), 16, 1.0, 1e6, kappa=1.0, u_rad=1e-7)
    fields = [0.3 * rng.uniform(-1, 1, (n, n, n)) for _ in range(3)] + \
             [1e-3 * rng.normal(size=(n, n, n)) for _ in range(3)] + [np.exp(0.3 * rng.normal(size=(n, n, n)))]
    x, y, z = (rng.uniform(-1, 1, 300) for _ in range(3))
    chi = rng.uniform(0.5, 1.5, (300, 16))
    dt = 0.05
    a = orc.step(prm, fields, x, y, z, dt, chi, nthreads=1)
    b = orc.step(prm, fields, x, y, z, dt, chi, nthreads=4)
    for u, v in zip(a, b):
        assert np.array_equal(u, v)
    k1, rho_old, xs = orc.push_stage0(prm, fields, x, y, z, dt)
    x1, y1, z1, st = orc.push_stage1(prm, fields, x, y, z, xs, k1, dt)
    chi1, nsub, lost = orc.spectral_update(prm, fields, x1, y1, z1, rho_old, dt, chi)
    assert np.array_equal(a[0], x1) and np.array_equal(a[3], chi1) and np.array_equal(a[4], nsub)
