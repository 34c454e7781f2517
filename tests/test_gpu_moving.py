"""GPU parity of the per-particle moving energy grid (lp_bind_energy_grid, lp_moving.cu; NEXT-5, readings E1-E4)
against oracle/orc_moving_update: edges and spectra elementwise within 1e-10 relative (positions bit for bit),
at all six bin counts, staged and through lp_step with re-sorts, plus the two laws north_star names."""
import numpy as np
import pytest
import torch

import lp_inputs as I
import paper_2602_23434_b200 as P
from oracle import lp_oracle as orc
from lp_testlib import assert_chi_close, fields_to_numpy, oracle_params, u_rad_of

pytestmark = pytest.mark.gpu
B = P.binding


def host(t):
    return t.detach().cpu().numpy()


def setup(w, pingpong=False):
    fields = I.make_fields(w, device="cpu")
    u_rad = u_rad_of(w, fields)
    x, y, z, pid = I.make_particles(w, shuffle_ids=True)
    chi = I.make_spectrum(w)
    lp = P.LP(P.config_from_workload(w, u_rad=u_rad))
    lp.set_fields(fields)
    lp.bind_particles(x, y, z, pid, chi)
    lp.bind_diag(nsub=True, lost=False)
    lp.bind_energy_grid()
    if pingpong:
        lp.set_pingpong(True)
    E, dE, Ec = orc.bin_table(w.nbins, w.e_min, w.e_max)
    return lp, oracle_params(w, u_rad), fields_to_numpy(fields), [x, y, z, pid, chi, np.tile(E, (w.np, 1))]


def oracle_step(prm, f_np, st, dt, sort):
    x, y, z, pid, chi, eng = st
    if sort:
        perm = orc.sort_perm(orc.cell_key(prm, x, y, z), pid)
        x, y, z, pid, chi, eng = x[perm], y[perm], z[perm], pid[perm], chi[perm], eng[perm]
    k1, rho_old, xs = orc.push_stage0(prm, f_np, x, y, z, dt, nthreads=8)
    x, y, z, status = orc.push_stage1(prm, f_np, x, y, z, xs, k1, dt, nthreads=8)
    eng, chi = orc.moving_update(prm, f_np, x, y, z, rho_old, dt, eng, chi, nthreads=8)
    return [x, y, z, pid, chi, eng]


def check(lp, st):
    n = st[0].shape[0]
    assert np.array_equal(host(lp.id)[:n].view(np.uint64), st[3])
    for g, w in zip((lp.x, lp.y, lp.z), st[:3]):
        assert np.array_equal(host(g)[:n], w)
    assert_chi_close(host(lp.eng)[:n], st[5], what="eng")
    assert_chi_close(host(lp.chi)[:n], st[4])
    assert (host(lp.nsub)[:n] == 1).all()


@pytest.mark.parametrize("nbins,np_", [(16, 3000 + 5), (32, 2000 + 31), (64, 4097), (128, 1500), (256, 777), (512, 300 + 33)])
def test_moving_grid_staged_matches_oracle(nbins, np_):
    w = I.workload(3).scaled(n=12, np=np_, nbins=nbins, sort_every=0)
    lp, prm, f_np, st = setup(w)
    for _ in range(3):
        lp.push(w.dt, 0)
        lp.push(w.dt, 1)
        lp.spectral_update(w.dt)
        st = oracle_step(prm, f_np, st, w.dt, False)
    check(lp, st)
    d = lp.diag()
    want = float(np.sum(st[4] * np.diff(st[5], axis=1)))
    assert abs(d["number"] - want) <= 1e-12 * abs(want) and d["max_substeps"] == 1
    # every bin keeps its number (E3): compare with the initial spectrum on the fixed table
    E, dE, Ec = orc.bin_table(w.nbins, w.e_min, w.e_max)
    chi0 = I.make_spectrum(w)
    pid0 = I.make_particles(w, shuffle_ids=True)[3]
    order = np.argsort(pid0); back = np.argsort(st[3])
    n_now = (host(lp.chi) * np.diff(host(lp.eng), axis=1))[back]
    assert np.allclose(n_now, (chi0 * dE[None, :])[order], rtol=1e-11, atol=0)


@pytest.mark.parametrize("pingpong", [False, True])
@pytest.mark.parametrize("nbins,np_", [(64, 6000 + 3), (16, 2500), (256, 999)])
def test_moving_grid_lp_step_with_resort(nbins, np_, pingpong):
    w = I.workload(3).scaled(n=12, np=np_, nbins=nbins, sort_every=2)
    lp, prm, f_np, st = setup(w, pingpong)
    for k in range(5):
        lp.step(w.dt)
        st = oracle_step(prm, f_np, st, w.dt, k % 2 == 0)
    check(lp, st)
    lp.sort()
    perm = orc.sort_perm(orc.cell_key(prm, *st[:3]), st[3])
    st = [a[perm] for a in st]
    check(lp, st)
    if pingpong:                                         # leaving ping-pong brings state and grid home
        lp.set_pingpong(False)
        assert lp.eng.data_ptr() == lp._eng.data_ptr() and lp.x.data_ptr() == lp._bound[0].data_ptr()
        check(lp, st)
        lp.step(w.dt)                                    # step 6: no re-sort due
        check(lp, oracle_step(prm, f_np, st, w.dt, False))


def test_moving_grid_synchrotron_law_and_unsupported_calls():
    """Workload 1 (uniform B, v = 0): after 100 lp_step every edge is E0 / (1 + c_r E0 t) (north_star)."""
    w = I.workload(1)
    E = I.bin_edges(w.nbins, w.e_min, w.e_max)
    cr = w.kappa * 0.5 * w.b0 ** 2
    dt = 0.9 * w.cfl_e / (cr * E[-2] ** 2 / (E[-1] - E[-2]))
    lp, prm, f_np, st = setup(w)
    for _ in range(100):
        lp.step(dt)
    eng = host(lp.eng)
    assert np.allclose(eng, (E / (1.0 + cr * E * dt * 100))[None, :], rtol=1e-12, atol=0)
    hx = torch.zeros(w.np, dtype=torch.float64).pin_memory()
    with pytest.raises(B.LPError) as e:
        lp.step_host(dt, hx, hx, hx, torch.zeros(w.np, dtype=torch.int64).pin_memory(),
                     torch.zeros((w.np, w.nbins), dtype=torch.float64).pin_memory())
    assert e.value.status == B.LP_ERR_UNSUPPORTED
    lp.unbind_energy_grid()
    lp.step(dt)                                  # back on the fixed bins
    assert lp.diag()["max_substeps"] >= 1


def test_sort_without_scratch_is_refused():
    w = I.workload(3).scaled(n=8, np=500, nbins=32, sort_every=0)
    fields = I.make_fields(w, device="cpu")
    x, y, z, pid = I.make_particles(w)
    lp = P.LP(P.config_from_workload(w, u_rad=0.0))
    lp.set_fields(fields)
    lp.bind_particles(x, y, z, pid, I.make_spectrum(w))
    lp.bind_energy_grid(sortable=False)
    with pytest.raises(B.LPError) as e:
        lp.sort()
    assert e.value.status == B.LP_ERR_STATE


def test_grid_rows_travel_with_their_particles():
    """Compaction, the exchange and growth move the energy-grid rows with the particles: the oracle's
    orc_compact / orc_migrate_* are run on rows that are chi and eng side by side (they move "every parameter"
    of a particle, whatever its width)."""
    rng = np.random.default_rng(9)
    n, nb = 3000, 32
    w = I.workload(3).scaled(n=12, np=n, nbins=nb, sort_every=0)
    lp, prm, f_np, st = setup(w)
    for _ in range(2):                                   # give every particle its own grid
        lp.step(w.dt)
        st = oracle_step(prm, f_np, st, w.dt, False)
    check(lp, st)
    x, y, z, pid, chi, eng = st
    wide = np.concatenate([chi, eng], axis=1)            # [n][2 nb + 1]

    def split(rows):
        return rows[:, :nb], rows[:, nb:]

    # deletion with hole filling
    flag = (rng.uniform(size=n) < 0.3).astype(np.int32)
    n1 = lp.compact(torch.from_numpy(flag).to(lp.device))
    x, y, z, pid, wide = orc.compact(flag, x, y, z, pid, wide)
    chi, eng = split(wide)
    check(lp, [x, y, z, pid, chi, eng])
    assert n1 == x.shape[0]

    # one directional exchange: this rank owns x in [-1, 0.2); what leaves comes back as "arrivals" from the
    # other side with shifted ids (a stand-in for the neighbour)
    nl, nr = lp.migrate_count(0, -1.0, 0.2)
    assert B.lp_migrate_record_bytes(lp.ctx) == 32 + 8 * nb + 8 * (nb + 1)
    bl, br = lp.migrate_pack(nl, nr)
    dest, holes, left, right = orc.migrate_pack(0, -1.0, 0.2, -1.0, 1.0, 1, x, y, z, pid, wide)
    assert (nl, nr) == (left[0].shape[0], right[0].shape[0]) and nr > 0
    raw = br.cpu().numpy()[: nr * (32 + 8 * nb + 8 * (nb + 1))]
    d = raw.view(np.float64)
    assert np.array_equal(d[:nr], right[0]) and np.array_equal(raw.view(np.uint64)[3 * nr:4 * nr], right[3])
    assert_chi_close(d[4 * nr:4 * nr + nr * nb].reshape(nr, nb), right[4][:, :nb])       # (spectra: 1e-10, not bits)
    assert_chi_close(d[4 * nr + nr * nb:].reshape(nr, nb + 1), right[4][:, nb:], what="eng")
    lp.reserve(nr, e=8)                                  # grow between pack and unpack: the grid follows
    n2 = lp.migrate_unpack(br, nr, bl, nl)               # the leavers come back in (right buffer first)
    x, y, z, pid, wide = orc.migrate_unpack(holes, right, left, x, y, z, pid, wide)
    chi, eng = split(wide)
    assert n2 == x.shape[0]
    check(lp, [x, y, z, pid, chi, eng])
    lp.step(w.dt)                                        # and the moving-grid update goes on
    check(lp, oracle_step(prm, f_np, [x, y, z, pid, chi, eng], w.dt, False))


@pytest.mark.parametrize("nbins", [16, 64, 128, 512])
def test_shock_update_on_the_moving_grid(nbins):
    """lp_shock_update with a bound grid: every flagged row on its own edges, against orc_shock_update_grid."""
    w = I.workload(3).scaled(n=12, np=1500 + 7, nbins=nbins, sort_every=0)
    lp, prm, f_np, st = setup(w)
    for _ in range(3):                                   # grids that differ from particle to particle
        lp.step(w.dt)
        st = oracle_step(prm, f_np, st, w.dt, False)
    rng = np.random.default_rng(nbins)
    r = np.where(rng.uniform(size=w.np) < 0.6, rng.uniform(1.5, 4.0, size=w.np), 1.0)
    r[::53] = np.nan
    lp.shock_update(torch.from_numpy(r).to(lp.device), 0.05)
    before = st[4].copy()
    st[4] = orc.shock_update_grid(st[5], r, 0.05, st[4])
    check(lp, st)
    untouched = ~(r > 1.0)
    got = host(lp.chi)
    assert_chi_close(got[untouched], before[untouched])
    wdt = np.diff(host(lp.eng), axis=1)
    assert np.allclose((got * wdt).sum(axis=1), (before * np.diff(st[5], axis=1)).sum(axis=1), rtol=1e-12, atol=0)
