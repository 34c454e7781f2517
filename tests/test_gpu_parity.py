"""GPU parity tests: the CUDA path (through the C ABI) against the CPU oracle on the same seeded
inputs, element by element.  Bit-exact for keys, sort order, gathered values and positions
(R14); relative 1e-10 for spectra; n_sub compared exactly."""
import numpy as np
import pytest
import torch

import lp_inputs as I
import paper_2602_23434_b200 as P
from oracle import lp_oracle as orc

from lp_testlib import (REL_TOL, assert_chi_close, assert_nsub_equal, fields_to_numpy, oracle_params,
                        oracle_sort_state, u_rad_of, workload1_dt)

pytestmark = pytest.mark.gpu
B = P.binding


def small_turbulent(n=12, np_=1000 + 37, nbins=64, sort_every=0, **kw):
    return I.workload(3).scaled(n=n, np=np_, nbins=nbins, sort_every=sort_every, **kw)


DIAG_KINDS = ("full", "nsub")      # "nsub": no `lost` output bound = the DIAG=false kernels (what bench.py times)


def setup_pair(w, shuffle_ids=False, diag="full", jitter=True, pingpong=False):
    """Returns (lp, prm, fields_np, x, y, z, pid, chi) with the GPU side bound to copies.
    diag: "full" binds n_sub and lost (the DIAG=true kernel instantiations), "nsub" binds n_sub only
    (lp_api.cu picks DIAG=false when no `lost` output is bound: the instantiations bench.py times), None
    binds nothing.  pingpong: re-sorts leave the state in the workspace twins of the bound arrays
    (lp_set_pingpong); lp.x, lp.chi ... follow it."""
    fields = I.make_fields(w, device="cpu")
    u_rad = u_rad_of(w, fields)
    f_np = fields_to_numpy(fields)
    x, y, z, pid = I.make_particles(w, shuffle_ids=shuffle_ids)
    chi = I.make_spectrum(w, jitter=jitter)
    lp = P.LP(P.config_from_workload(w, u_rad=u_rad))
    lp.set_fields(fields)
    lp.bind_particles(x, y, z, pid, chi)
    if diag:
        lp.bind_diag(nsub=True, lost=(diag == "full"))
    if pingpong:
        lp.set_pingpong(True)
    return lp, oracle_params(w, u_rad), f_np, x, y, z, pid, chi


def host(t):
    return t.detach().cpu().numpy()


# ------------------------------------------------------------------ a1, a4: key and gather

@pytest.mark.parametrize("periodic", [(1, 1, 1), (0, 0, 0), (1, 0, 1)])
def test_key_and_gather_bit_exact(periodic):
    w = small_turbulent(np_=4096 + 5, periodic=periodic)
    lp, prm, f_np, x, y, z, pid, chi = setup_pair(w)
    # put some particles on faces, on the domain edges and slightly outside
    x[:8] = [-1.0, 1.0 - 1e-16, -1.0 + 2.0 / w.n, 0.0, 1.0, -1.0000001, 0.999999999, -0.5]
    y[:4] = [-1.0, 0.0, 1.0 / 3.0, -1.0 + 2.0 / w.n * 5]
    lp.bind_particles(x, y, z, pid, chi)
    out7, key = lp.interpolate()
    torch.cuda.synchronize()
    want_key = orc.cell_key(prm, x, y, z)
    assert np.array_equal(host(key).view(np.uint32), want_key)
    want = orc.gather(prm, f_np, x, y, z)
    assert np.array_equal(host(out7), want), "gather not bit-identical: max abs diff %g" % np.max(np.abs(host(out7) - want))


def test_key_non_cubic_grid():
    cfg = P.make_config(5, 7, 3, (-1, 0, 2), (1, 3.5, 2.75), (1, 1, 1), 500, 16, 1.0, 1e4)
    rng = np.random.default_rng(0)
    x = rng.uniform(-1, 1, 500); y = rng.uniform(0, 3.5, 500); z = rng.uniform(2, 2.75, 500)
    lp = P.LP(cfg)
    lp.bind_particles(x, y, z, np.arange(500, dtype=np.uint64), np.ones((500, 16)))
    _, key = lp.interpolate(want_fields=False)
    prm = orc.make_params(5, 7, 3, (-1, 0, 2), (1, 3.5, 2.75), (1, 1, 1), 16, 1.0, 1e4)
    assert np.array_equal(host(key).view(np.uint32), orc.cell_key(prm, x, y, z))
    f = [rng.normal(size=(3, 7, 5)) for _ in range(7)]
    lp.set_fields([torch.from_numpy(a) for a in f])
    out7, _ = lp.interpolate(want_key=False)
    assert np.array_equal(host(out7), orc.gather(prm, f, x, y, z))


# ------------------------------------------------------------------ a5, a6: push

@pytest.mark.parametrize("periodic", [(1, 1, 1), (0, 0, 0), (1, 0, 1)])
@pytest.mark.parametrize("np_,n", [(6000 + 3, 12), (70001, 40), (31, 6)])
def test_interpolate_tiled_bit_exact(periodic, np_, n):
    """The shared-memory-tile gather gives lp_interpolate's bits: sorted by cell (tiles), then shuffled (the
    blocks fall back to the direct gather), with far-away particles in one block."""
    w = small_turbulent(n=n, np_=np_, periodic=periodic)
    lp, prm, f_np, x, y, z, pid, chi = setup_pair(w, shuffle_ids=True)
    want = orc.gather(prm, f_np, x, y, z)
    assert np.array_equal(host(lp.interpolate_tiled()), want)            # unsorted: most blocks fall back
    lp.sort()
    order = np.argsort(host(lp.id).view(np.uint64)); inv = np.argsort(np.argsort(pid))
    got = host(lp.interpolate_tiled())[:, order][:, inv]
    assert np.array_equal(got, want)                                     # sorted: tiles
    direct, _ = lp.interpolate(want_key=False)
    assert np.array_equal(host(direct), host(lp.interpolate_tiled()))
    if np_ > 100:                                                        # a few particles far outside the box
        lp.x[:5] = torch.tensor([1e3, -1e3, 7.5, 1e12, -3.0], dtype=torch.float64, device=lp.device)
        direct, _ = lp.interpolate(want_key=False)
        assert np.array_equal(host(direct), host(lp.interpolate_tiled()), equal_nan=True)


@pytest.mark.parametrize("periodic", [(1, 1, 1), (0, 0, 0)])
def test_push_positions_bit_exact_over_steps(periodic):
    w = small_turbulent(np_=3000 + 11, periodic=periodic)
    lp, prm, f_np, x, y, z, pid, chi = setup_pair(w)
    dt = w.dt * 3.0          # large steps: many wraps on the periodic box
    for _ in range(25):
        lp.push(dt, 0)
        lp.push(dt, 1)
        k1, rho_old, xs = orc.push_stage0(prm, f_np, x, y, z, dt)
        x, y, z, st = orc.push_stage1(prm, f_np, x, y, z, xs, k1, dt)
    torch.cuda.synchronize()
    assert np.array_equal(host(lp.x), x) and np.array_equal(host(lp.y), y) and np.array_equal(host(lp.z), z)
    if periodic == (1, 1, 1):
        assert (x >= -1).all() and (x < 1).all()
    d = lp.diag()
    assert d["n_outside"] == 0 or periodic != (1, 1, 1)


# ------------------------------------------------------------------ a2: sort

@pytest.mark.parametrize("pingpong", [False, True])
@pytest.mark.parametrize("np_,id_shift", [(1, 33), (31, 33), (4097, 33), (50000, 33), (5003, 62)])
def test_sort_order_and_permutation_bit_exact(np_, id_shift, pingpong):
    """ids wider than 32 bits (35 and 64 significant bits: five and eight radix passes over the ids)."""
    w = small_turbulent(n=6, np_=np_, nbins=16)          # 216 cells: many ties per key
    lp, prm, f_np, x, y, z, pid, chi = setup_pair(w, shuffle_ids=True)
    pid = pid + np.uint64(1 << id_shift) * (pid % np.uint64(3))
    lp.bind_particles(x, y, z, pid, chi)
    lp.set_pingpong(pingpong)
    lp.sort()
    torch.cuda.synchronize()
    sx, sy, sz, sid, schi, skey, perm = oracle_sort_state(prm, x, y, z, pid, chi)
    assert np.array_equal(host(lp.id).view(np.uint64), sid)
    assert np.array_equal(host(lp.x), sx) and np.array_equal(host(lp.y), sy) and np.array_equal(host(lp.z), sz)
    assert np.array_equal(host(lp.chi), schi)
    _, key = lp.interpolate(want_fields=False)
    assert np.array_equal(host(key).view(np.uint32), skey)


# ------------------------------------------------------------------ a7-a10: spectral update

@pytest.mark.parametrize("diag", DIAG_KINDS)
@pytest.mark.parametrize("nbins", [16, 32, 64, 128, 256, 512])
def test_spectral_update_matches_oracle(nbins, diag):
    # e range of workload 5 and a strong field: n_sub spans 1 (16 bins) to O(10^2..10^3) (512 bins),
    # all below the cap (a capped row violates the CFL bound and is compared separately below)
    w = small_turbulent(np_=2000 + 45, nbins=nbins, e_min=1.0, e_max=1e8, brms=3e-3)
    lp, prm, f_np, x, y, z, pid, chi = setup_pair(w, diag=diag)
    dt = 0.005
    lp.push(dt, 0); lp.push(dt, 1); lp.spectral_update(dt)
    k1, rho_old, xs = orc.push_stage0(prm, f_np, x, y, z, dt)
    x1, y1, z1, st = orc.push_stage1(prm, f_np, x, y, z, xs, k1, dt)
    chi1, nsub, lost = orc.spectral_update(prm, f_np, x1, y1, z1, rho_old, dt, chi, nthreads=8)
    torch.cuda.synchronize()
    assert np.array_equal(host(lp.x), x1)
    assert (nsub > 0).all(), "test set-up: no row may hit the substep cap here"
    assert_nsub_equal(host(lp.nsub), nsub, "(nbins=%d)" % nbins)
    assert_chi_close(host(lp.chi), chi1)
    E, dE, _ = orc.bin_table(nbins, w.e_min, w.e_max)
    number = chi @ dE
    if diag == "full":
        assert np.max(np.abs(host(lp.lost) - lost) / number) < REL_TOL
    if nbins >= 256:
        assert nsub.max() > 1
    # the library's bin table against the oracle's
    Eg, dEg = lp.bins()
    assert np.max(np.abs(Eg / E - 1)) < 1e-15 and np.max(np.abs(dEg / dE - 1)) < 1e-13


def test_spectral_update_sign_changing_advection_and_cap():
    """Strong compression/expansion (a of both signs) with losses; and the n_sub cap."""
    w = small_turbulent(np_=3000, nbins=64, sigma_rho=2.0, brms=1e-3, max_substeps=12)
    lp, prm, f_np, x, y, z, pid, chi = setup_pair(w)
    dt = 4 * w.dt
    lp.push(dt, 0); lp.push(dt, 1); lp.spectral_update(dt)
    x1, y1, z1, chi1, nsub, lost, st = orc.step(prm, f_np, x, y, z, dt, chi, nthreads=8)
    torch.cuda.synchronize()
    assert (nsub < 0).any() and (nsub > 0).any()           # some capped, some not
    assert_nsub_equal(host(lp.nsub), nsub)
    capped = nsub < 0
    assert_chi_close(host(lp.chi)[~capped], chi1[~capped])
    # capped rows violate the CFL bound: the scheme is unstable there (chi changes sign, rounding is
    # amplified), so they are compared against the row's scale instead of element by element
    gc, oc = host(lp.chi)[capped], chi1[capped]
    assert np.all(np.abs(gc - oc) <= 1e-8 * np.abs(oc).max(axis=1, keepdims=True))
    d = lp.diag()
    assert d["n_capped"] == int(capped.sum()) and d["max_substeps"] == 12
    assert d["sum_substeps"] == int(np.abs(nsub).sum())
    # The compare of the capped rows above is a sanity check (same order of magnitude, no garbage), not a parity
    # claim: such rows are outside the method.  A caller who wants them to be an error gets one:
    B.lp_set_cap_policy(lp.ctx, True)
    with pytest.raises(B.LPError) as e:
        lp.diag()
    assert e.value.status == B.LP_ERR_UNSUPPORTED and "max_substeps" in str(e.value)
    B.lp_set_cap_policy(lp.ctx, False)
    assert lp.diag()["n_capped"] == int(capped.sum())


def test_number_conservation_diag():
    w = small_turbulent(np_=5000, nbins=128)
    lp, prm, f_np, x, y, z, pid, chi = setup_pair(w)
    n0 = lp.diag()["number"]
    E, dE, _ = orc.bin_table(w.nbins, w.e_min, w.e_max)
    assert abs(n0 / float((chi @ dE).sum()) - 1) < 1e-12
    lp.step(w.dt)
    d = lp.diag()
    assert abs((d["number"] + d["lost"]) / n0 - 1) < 1e-12
    assert d["steps"] == 1 and d["sorts"] == 0


# ------------------------------------------------------------------ third-order pusher (NEXT-4)

@pytest.mark.parametrize("periodic", [(1, 1, 1), (0, 1, 0)])
def test_push_rk3_bit_exact_and_spectral_update_follows(periodic):
    """lp_push_rk3 stage by stage vs the oracle (positions of every stage bit for bit, outside flags),
    fields changed between the stages, then lp_spectral_update with the rho_old of stage 0."""
    w = small_turbulent(np_=4000 + 5, nbins=32).scaled(periodic=periodic, dt=0.05)
    lp, prm, f_np, x, y, z, pid, chi = setup_pair(w)
    fields_b = I.make_fields(w.scaled(seed=w.seed + 1), device="cpu")          # "advanced" fields for stages 1, 2
    fb_np = fields_to_numpy(fields_b)
    for step in range(3):
        xe, ye, ze, rho_old, st, mids = orc.push_rk3(prm, [f_np, fb_np, fb_np], x, y, z, w.dt)
        lp.set_fields([f.cuda() for f in I.make_fields(w, device="cpu")])
        lp.push_rk3(w.dt, 0)
        assert np.array_equal(host(lp.x), mids[0][0]) and np.array_equal(host(lp.z), mids[0][2])
        lp.set_fields([f.cuda() for f in fields_b])
        lp.push_rk3(w.dt, 1)
        assert np.array_equal(host(lp.x), mids[1][0]) and np.array_equal(host(lp.y), mids[1][1])
        lp.push_rk3(w.dt, 2)
        assert np.array_equal(host(lp.x), xe) and np.array_equal(host(lp.y), ye) and np.array_equal(host(lp.z), ze)
        lp.spectral_update(w.dt)
        chi, nsub, lost = orc.spectral_update(prm, fb_np, xe, ye, ze, rho_old, w.dt, chi, nthreads=8)
        assert_nsub_equal(host(lp.nsub), nsub)
        assert_chi_close(host(lp.chi), chi)
        assert lp.diag()["n_outside"] == int((st != 0).sum())
        x, y, z = xe, ye, ze
    with pytest.raises(P.binding.LPError):
        lp.push_rk3(w.dt, 2)                               # stages out of order


# ------------------------------------------------------------------ shock crossing (Eq. 7-8, NEXT-1)

@pytest.mark.parametrize("nbins", [16, 32, 64, 128, 256, 512])
def test_shock_update_matches_oracle(nbins):
    """lp_shock_update vs the oracle row by row: flagged rows (r > 1) to 1e-10 relative, unflagged rows
    (r <= 1, NaN) bit for bit untouched, empty bins below the lowest occupied one stay exactly zero."""
    w = small_turbulent(np_=3000 + 37, nbins=nbins)
    lp, prm, f_np, x, y, z, pid, chi = setup_pair(w)
    rng = np.random.default_rng(nbins)
    r = rng.uniform(1.5, 4.0, w.np)
    r[rng.uniform(size=w.np) < 0.4] = 1.0                     # no shock
    r[::97] = np.nan
    r[5] = 0.3
    chi = chi.copy()
    chi[::7, : nbins // 4] = 0.0                              # rows with an empty low end
    chi[11, :] = 0.0                                          # an empty row
    lp.chi.copy_(torch.from_numpy(chi))
    E, dE, _ = orc.bin_table(w.nbins, w.e_min, w.e_max)
    q_r = 0.05
    expect = orc.shock_update(E, dE, r, q_r, chi)
    lp.shock_update(torch.from_numpy(r).cuda(), q_r)
    torch.cuda.synchronize()
    got = host(lp.chi)
    untouched = ~(r > 1.0)
    assert np.array_equal(got[untouched], chi[untouched]) and np.array_equal(got[11], chi[11])
    assert_chi_close(got, expect)
    assert np.array_equal(got == 0.0, expect == 0.0)
    num_in, num_out = (chi * dE).sum(axis=1), (got * dE).sum(axis=1)
    ok = num_in > 0
    assert np.max(np.abs(num_out[ok] / num_in[ok] - 1)) < 1e-13                  # number conserved per row


# ------------------------------------------------------------------ deletion + hole filling (NEXT-2)

@pytest.mark.parametrize("np_,frac", [(1, 1.0), (33, 0.5), (5000 + 7, 0.05), (70001, 0.3), (4097, 0.0), (4097, 1.0)])
def test_compact_matches_oracle_bit_exact(np_, frac):
    """lp_compact vs the paper's five steps in the oracle: the same particles in the same slots, every
    parameter bit for bit; the context then steps the shortened set like the oracle does."""
    w = small_turbulent(np_=np_, nbins=32)
    lp, prm, f_np, x, y, z, pid, chi = setup_pair(w, shuffle_ids=True)
    rng = np.random.default_rng(np_)
    flag = (rng.uniform(size=np_) < frac).astype(np.int32)
    n_new = lp.compact(torch.from_numpy(flag).cuda())
    x, y, z, pid, chi = orc.compact(flag, x, y, z, pid, chi)
    assert n_new == x.shape[0] == np_ - int(flag.sum()) and lp.diag()["np"] == n_new
    assert np.array_equal(host(lp.id)[:n_new].view(np.uint64), pid)
    assert np.array_equal(host(lp.x)[:n_new], x) and np.array_equal(host(lp.y)[:n_new], y)
    assert np.array_equal(host(lp.z)[:n_new], z) and np.array_equal(host(lp.chi)[:n_new], chi)
    if n_new:
        lp.step(w.dt)
        x, y, z, chi, nsub, lost, st = orc.step(prm, f_np, x, y, z, w.dt, chi, nthreads=8)
        assert np.array_equal(host(lp.x)[:n_new], x)
        assert_nsub_equal(host(lp.nsub)[:n_new], nsub)
        assert_chi_close(host(lp.chi)[:n_new], chi)


def test_compact_outflow_deletes_what_left_the_box():
    """Open (zero-gradient) box: after a step some particles are outside; lp_compact without flags deletes
    exactly those (Particles_Boundary) and a second call without a new push is refused."""
    w = small_turbulent(np_=6000, nbins=16).scaled(periodic=(0, 0, 0), dt=0.2)
    lp, prm, f_np, x, y, z, pid, chi = setup_pair(w)
    lp.step(w.dt)
    x, y, z, chi, nsub, lost, st = orc.step(prm, f_np, x, y, z, w.dt, chi, nthreads=8)
    assert (st != 0).sum() > 10
    n_new = lp.compact()
    x, y, z, pid, chi = orc.compact((st != 0).astype(np.int32), x, y, z, pid, chi)
    assert n_new == x.shape[0]
    assert np.array_equal(host(lp.id)[:n_new].view(np.uint64), pid) and np.array_equal(host(lp.x)[:n_new], x)
    assert_chi_close(host(lp.chi)[:n_new], chi)            # (rows went through one update: 1e-10, not bits)
    with pytest.raises(P.binding.LPError):
        lp.compact()


def test_injection_within_capacity():
    """Particles are injected by writing them behind the current ones and raising the count
    (lp_set_count): a step on the first 3000, then on all 5000."""
    w = small_turbulent(np_=5000, nbins=32)
    lp, prm, f_np, x, y, z, pid, chi = setup_pair(w)
    n0 = 3000
    lp.set_count(n0)
    lp.step(w.dt)
    xa, ya, za, chia, nsub, lost, st = orc.step(prm, f_np, x[:n0], y[:n0], z[:n0], w.dt, chi[:n0], nthreads=8)
    assert lp.diag()["np"] == n0
    assert np.array_equal(host(lp.x)[:n0], xa) and np.array_equal(host(lp.x)[n0:], x[n0:])      # the tail is untouched
    assert np.array_equal(host(lp.chi)[n0:], chi[n0:])
    lp.set_count(w.np)
    lp.step(w.dt)
    x2 = np.concatenate([xa, x[n0:]]); y2 = np.concatenate([ya, y[n0:]]); z2 = np.concatenate([za, z[n0:]])
    chi2 = np.concatenate([chia, chi[n0:]])
    xb, yb, zb, chib, nsub, lost, st = orc.step(prm, f_np, x2, y2, z2, w.dt, chi2, nthreads=8)
    assert np.array_equal(host(lp.x), xb) and np.array_equal(host(lp.z), zb)
    assert_nsub_equal(host(lp.nsub), nsub)
    assert_chi_close(host(lp.chi), chib)
    with pytest.raises(P.binding.LPError):
        lp.set_count(w.np + 1)


# ------------------------------------------------------------------ whole step, with re-sort

@pytest.mark.parametrize("pingpong", [False, True])
@pytest.mark.parametrize("diag", DIAG_KINDS)
@pytest.mark.parametrize("nbins,np_", [(64, 6000 + 3), (16, 2500), (128, 1500), (32, 4097), (256, 999), (512, 700)])
def test_lp_step_with_resort_matches_oracle(nbins, np_, diag, pingpong):
    """Eight fused steps with a re-sort every third.  pingpong: the re-sort is folded into the fused kernel
    (rows, positions and ids read through the permutation, written to the other buffer set)."""
    w = small_turbulent(n=10, np_=np_, nbins=nbins, sort_every=3)
    lp, prm, f_np, x, y, z, pid, chi = setup_pair(w, shuffle_ids=True, diag=diag, pingpong=pingpong)
    dt = w.dt
    for s in range(8):
        lp.step(dt)
        if s % 3 == 0:
            x, y, z, pid, chi, _, _ = oracle_sort_state(prm, x, y, z, pid, chi)
        x, y, z, chi, nsub, lost, st = orc.step(prm, f_np, x, y, z, dt, chi, nthreads=8)
    torch.cuda.synchronize()
    assert np.array_equal(host(lp.id).view(np.uint64), pid)       # same order => compare in place
    assert np.array_equal(host(lp.x), x) and np.array_equal(host(lp.z), z)
    assert_nsub_equal(host(lp.nsub), nsub)
    assert_chi_close(host(lp.chi), chi)
    d = lp.diag()
    assert d["steps"] == 8 and d["sorts"] == 3
    if pingpong:
        # three re-sorts: the state is in the workspace twins now; switching ping-pong off brings it home
        bound = lp._bound
        assert lp.x.data_ptr() != bound[0].data_ptr()
        lp.set_pingpong(False)
        torch.cuda.synchronize()
        assert lp.x.data_ptr() == bound[0].data_ptr()
        assert np.array_equal(host(bound[0]), x) and np.array_equal(host(bound[3]).view(np.uint64), pid)
        assert_chi_close(host(bound[4]), chi)


@pytest.mark.parametrize("np_,nbins,sort_every,diag", [
    (4000, 32, 0, "full"), (70001, 16, 0, "full"), (66000, 64, 2, "full"),
    # what bench.py's e2e leg runs: no diagnostics bound at all (DIAG=false kernels), and batch tails that are
    # not multiples of 32 at the bin counts with several ring slots per chunk
    (66000, 64, 2, None), (65536 + 1, 128, 0, None), (65536 + 31, 256, 0, "nsub"), (65536 + 33, 128, 2, "nsub"),
    (65536 + 33, 512, 0, None), (66000, 64, 2, "pingpong"), (65536 + 33, 128, 1, "pingpong")])
def test_lp_step_host_roundtrip(np_, nbins, sort_every, diag):
    """lp_step on host buffers: whole-array path (small sets, re-sort steps) and the batched pipeline
    (>= 65536 particles: copy-in, kernels and copy-out overlap) must both give the oracle's step."""
    w = small_turbulent(np_=np_, nbins=nbins, sort_every=sort_every)
    pingpong = diag == "pingpong"
    diag = "nsub" if pingpong else diag
    lp, prm, f_np, x, y, z, pid, chi = setup_pair(w, shuffle_ids=True, diag=diag, pingpong=pingpong)
    hx, hy, hz = (torch.from_numpy(a.copy()).pin_memory() for a in (x, y, z))
    hid = torch.from_numpy(pid.view(np.int64).copy()).pin_memory()
    hchi = torch.from_numpy(chi.copy()).pin_memory()
    for s in range(2):                                   # with sort_every = 2: a re-sort step, then a pipelined one
        lp.step_host(w.dt, hx, hy, hz, hid, hchi)
        if sort_every and s % sort_every == 0:
            x, y, z, pid, chi, _, _ = oracle_sort_state(prm, x, y, z, pid, chi)
        x, y, z, chi, nsub, lost, st = orc.step(prm, f_np, x, y, z, w.dt, chi, nthreads=8)
    assert np.array_equal(hid.numpy().view(np.uint64), pid)
    assert np.array_equal(hx.numpy(), x) and np.array_equal(hy.numpy(), y) and np.array_equal(hz.numpy(), z)
    assert_chi_close(hchi.numpy(), chi)
    if diag:
        assert_nsub_equal(host(lp.nsub), nsub)
    assert lp.diag()["steps"] == 2


# ------------------------------------------------------------------ edge cases and error paths

@pytest.mark.parametrize("pingpong", [False, True])
def test_empty_and_tiny_particle_sets(pingpong):
    for n_p in (0, 1, 2, 33):
        w = small_turbulent(np_=n_p, nbins=16 if n_p % 2 else 64, sort_every=1)
        lp, prm, f_np, x, y, z, pid, chi = setup_pair(w, pingpong=pingpong)
        lp.step(w.dt)
        lp.step(w.dt)
        torch.cuda.synchronize()
        if n_p:
            for _ in range(2):
                x, y, z, pid, chi, _, _ = oracle_sort_state(prm, x, y, z, pid, chi)
                x, y, z, chi, nsub, lost, st = orc.step(prm, f_np, x, y, z, w.dt, chi)
            assert np.array_equal(host(lp.x), x)
            assert_chi_close(host(lp.chi), chi)
        assert lp.diag()["np"] == n_p


def test_state_errors():
    w = small_turbulent(np_=100)
    cfg = P.config_from_workload(w)
    lp = P.LP(cfg)
    with pytest.raises(B.LPError) as e:
        lp.step(0.1)                       # no particles bound
    assert e.value.status == B.LP_ERR_STATE
    x, y, z, pid = I.make_particles(w)
    lp.bind_particles(x, y, z, pid, I.make_spectrum(w))
    with pytest.raises(B.LPError) as e:
        lp.push(0.1, 0)                    # fields not set
    assert e.value.status == B.LP_ERR_STATE and "fields" in str(e.value)
    lp.set_fields(I.make_fields(w))
    with pytest.raises(B.LPError) as e:
        lp.push(0.1, 1)                    # stage 1 before stage 0
    assert e.value.status == B.LP_ERR_STATE
    with pytest.raises(B.LPError) as e:
        lp.spectral_update(0.1)            # needs rho_old of stage 0
    assert e.value.status == B.LP_ERR_STATE
    with pytest.raises(B.LPError) as e:
        lp.push(0.1, 2)
    assert e.value.status == B.LP_ERR_INVALID_ARG
    lp.push(0.1, 0)
    with pytest.raises(B.LPError) as e:
        lp.spectral_update(0.1)            # the push is not finished: x^{n+1} does not exist yet
    assert e.value.status == B.LP_ERR_STATE
    lp.push_rk3(0.1, 0); lp.push_rk3(0.1, 1)
    with pytest.raises(B.LPError) as e:
        lp.spectral_update(0.1)            # nor after two of three stages
    assert e.value.status == B.LP_ERR_STATE
    ctx2 = B.lp_create(cfg)
    with pytest.raises(B.LPError) as e:
        B.lp_bind_workspace(ctx2, lp.workspace.data_ptr() + 8, lp.workspace_bytes)
    assert e.value.status == B.LP_ERR_WORKSPACE
    with pytest.raises(B.LPError) as e:
        B.lp_bind_workspace(ctx2, lp.workspace.data_ptr() + (-lp.workspace.data_ptr()) % 256, 1024)
    assert e.value.status == B.LP_ERR_WORKSPACE
    B.lp_destroy(ctx2)
    lp.push(0.1, 0); lp.push(0.1, 1); lp.spectral_update(0.1)      # and the good order works
    torch.cuda.synchronize()
    assert lp.launch_count() >= 4


# ------------------------------------------------------------------ a8: substep count next to an integer

@pytest.mark.parametrize("nbins", [16, 64, 128, 512])
@pytest.mark.parametrize("diag", DIAG_KINDS)
def test_nsub_when_cfl_ratio_is_next_to_an_integer(nbins, diag):
    """dtau*lambda/C_E within the kernel's two-bin margin (>= 1e-12 relative) of an integer k: the kernel must
    then evaluate the other hull-vertex bins too and still return the oracle's full-scan integer.  Uniform
    fields (v = 0, rho = 1: a = 0, dtau = dt), dt chosen from the oracle's lambda so that the ratio is
    k (1 + eps), |eps| = 2e-13 or 5e-13: inside the margin, far outside the 1e-16 rounding of either side."""
    w = I.workload(1).scaled(n=4, np=257, nbins=nbins, e_min=1.0, e_max=1e8).scaled(b0=2e-3, support=None)
    lp, prm, f_np, x, y, z, pid, chi = setup_pair(w, diag=diag)
    E, dE, _ = orc.bin_table(nbins, w.e_min, w.e_max)
    cr = w.kappa * 0.5 * w.b0 ** 2
    _, lam = orc.cfl_nsub(E, dE, 0.0, cr, 1.0)
    for k in (1, 2, 7):
        for eps in (-5e-13, -2e-13, 2e-13, 5e-13):
            dt = k * (1.0 + eps) * w.cfl_e / lam
            lp.step(dt)
            x, y, z, chi, nsub, lost, st = orc.step(prm, f_np, x, y, z, dt, chi)       # (v = 0: nobody moves)
            assert set(np.unique(nsub)) <= {k, k + 1}
            assert_nsub_equal(host(lp.nsub), nsub, "(k=%d eps=%g)" % (k, eps))
            assert_chi_close(host(lp.chi), chi)


# ------------------------------------------------------------------ a2 after injection: ids wider than any bound id

@pytest.mark.parametrize("np_", [6000, 30000])
@pytest.mark.parametrize("pingpong", [False, True])
def test_sort_after_compaction_and_injection_of_wider_ids(pingpong, np_):
    """The number of radix passes over the ids must follow the ids that are there when the sort runs, not
    those bound at the start: delete some particles, inject new ones with ids far above every earlier id
    (more significant bits), raise the count, sort -- the order must be the oracle's (key, id) order.
    6000 particles on 216 cells stay inside the counting sort (at most 64 per cell); 30000 put about 139 in
    every cell, so the sort falls back to the radix passes, the one consumer of the measured id width."""
    w = small_turbulent(n=6, np_=np_, nbins=16)
    lp, prm, f_np, x, y, z, pid, chi = setup_pair(w, shuffle_ids=True, pingpong=pingpong)
    lp.sort()                                                     # a sort with the narrow ids first
    x, y, z, pid, chi, _, _ = oracle_sort_state(prm, x, y, z, pid, chi)
    rng = np.random.default_rng(7)
    flag = (rng.uniform(size=w.np) < 0.3).astype(np.int32)
    n_keep = lp.compact(torch.from_numpy(flag).cuda())
    x, y, z, pid, chi = orc.compact(flag, x, y, z, pid, chi)
    n_new = w.np - n_keep
    nx_, ny_, nz_ = (rng.uniform(-1, 1, n_new) for _ in range(3))
    nid = (np.uint64(1) << np.uint64(40)) + rng.permutation(n_new).astype(np.uint64) * np.uint64(1 << 20)
    nchi = rng.uniform(0.5, 1.5, (n_new, w.nbins))
    for t, a in ((lp.x, nx_), (lp.y, ny_), (lp.z, nz_), (lp.chi, nchi)):
        t[n_keep:] = torch.from_numpy(a).cuda()
    lp.id[n_keep:] = torch.from_numpy(nid.view(np.int64)).cuda()
    lp.set_count(w.np)
    x = np.concatenate([x, nx_]); y = np.concatenate([y, ny_]); z = np.concatenate([z, nz_])
    pid = np.concatenate([pid, nid]); chi = np.concatenate([chi, nchi])
    lp.sort()
    sx, sy, sz, sid, schi, skey, perm = oracle_sort_state(prm, x, y, z, pid, chi)
    assert np.array_equal(host(lp.id).view(np.uint64), sid)
    assert np.array_equal(host(lp.x), sx) and np.array_equal(host(lp.chi), schi)


@pytest.mark.parametrize("pingpong", [False, True])
def test_sort_with_duplicate_ids_loses_no_particle(pingpong):
    """Ids are unique by contract, but a caller's bug (an uninitialised tail after lp_set_count) must not cost a
    particle: with equal ids inside one cell the rank-counting sort used to write one slot of the permutation twice
    (round-2 advisor finding).  Such a set now goes through the stable radix passes: the result is ordered by
    (key, id) and is a permutation of what went in -- the order among equal pairs is not unique and not compared."""
    w = small_turbulent(n=6, np_=5000 + 1, nbins=16)
    lp, prm, f_np, x, y, z, pid, chi = setup_pair(w, shuffle_ids=True, pingpong=pingpong)
    key = orc.cell_key(prm, x, y, z)
    order = np.argsort(key, kind="stable")
    pid = pid.copy()
    for a, b in zip(order[:-1:7], order[1::7]):              # neighbours in key order: mostly the same cell
        if key[a] == key[b]:
            pid[b] = pid[a]
    assert len(np.unique(pid)) < w.np - 100
    chi[:, 0] = np.arange(w.np)                               # a tag that tells the rows apart
    lp.bind_particles(x, y, z, pid, chi)
    lp.sort()
    gid = host(lp.id).view(np.uint64); gx = host(lp.x); gchi = host(lp.chi)
    src = gchi[:, 0].astype(np.int64)
    assert np.array_equal(np.sort(src), np.arange(w.np))     # a permutation: nobody twice, nobody lost
    assert np.array_equal(gid, pid[src]) and np.array_equal(gx, x[src]) and np.array_equal(gchi, chi[src])
    gkey = key[src].astype(np.uint64)
    pairs = list(zip(gkey.tolist(), gid.tolist()))
    assert pairs == sorted(pairs)


# ------------------------------------------------------------------ seeded random configurations

@pytest.mark.parametrize("seed", range(24))
def test_random_small_configurations(seed):
    """Ragged sizes against the ring / chunk / batch boundaries of the kernels: random particle counts, bin
    counts, boundary kinds and re-sort periods; three fused steps, everything compared as in the other tests."""
    rng = np.random.default_rng(1000 + seed)
    np_ = int(rng.choice([1, 2, 31, 32, 33, 63, 65, 255, 257, 1023, 1025, 4095, 4129, int(rng.integers(1, 9000))]))
    nbins = int(rng.choice([16, 32, 64, 128, 256, 512]))
    periodic = tuple(int(v) for v in rng.integers(0, 2, 3))
    sort_every = int(rng.choice([0, 1, 2]))
    w = small_turbulent(n=int(rng.choice([4, 7, 12])), np_=np_, nbins=nbins, sort_every=sort_every).scaled(
        periodic=periodic, dt=float(rng.choice([0.01, 0.05])))
    lp, prm, f_np, x, y, z, pid, chi = setup_pair(w, shuffle_ids=True, diag=DIAG_KINDS[seed % 2],
                                                  pingpong=bool((seed // 2) % 2))
    for s in range(3):
        lp.step(w.dt)
        if sort_every and s % sort_every == 0:
            x, y, z, pid, chi, _, _ = oracle_sort_state(prm, x, y, z, pid, chi)
        x, y, z, chi, nsub, lost, st = orc.step(prm, f_np, x, y, z, w.dt, chi, nthreads=8)
    torch.cuda.synchronize()
    assert np.array_equal(host(lp.id).view(np.uint64), pid)
    assert np.array_equal(host(lp.x), x) and np.array_equal(host(lp.y), y) and np.array_equal(host(lp.z), z)
    assert_nsub_equal(host(lp.nsub), nsub)
    assert_chi_close(host(lp.chi), chi)
    d = lp.diag()
    assert d["n_outside"] == int((st != 0).sum()) and d["np"] == np_


# ------------------------------------------------------------------ several contexts at once

def test_two_contexts_from_two_host_threads():
    """lp.h: a context is used by one host thread at a time, but several contexts may run concurrently from
    different threads (they share no mutable state).  Two threads, each with its own context, bin count and
    stream, step at the same time; both must give the oracle's result."""
    import threading
    cases = [small_turbulent(np_=5000 + 3, nbins=64, sort_every=2), small_turbulent(np_=3000 + 1, nbins=256, sort_every=1, seed=99)]
    pairs = [setup_pair(w, shuffle_ids=True, diag="nsub", pingpong=(i == 1)) for i, w in enumerate(cases)]
    errors = []
    torch.cuda.synchronize()            # the set-up ran on the default stream

    def work(i):
        try:
            lp, w = pairs[i][0], cases[i]
            stream = torch.cuda.Stream()
            with torch.cuda.stream(stream):
                for _ in range(6):
                    lp.step(w.dt)
                stream.synchronize()
        except Exception as e:          # noqa: BLE001 -- reported by the main thread
            errors.append((i, e))

    threads = [threading.Thread(target=work, args=(i,)) for i in range(2)]
    for t in threads:
        t.start()
    for t in threads:
        t.join()
    assert not errors, errors
    torch.cuda.synchronize()
    for (lp, prm, f_np, x, y, z, pid, chi), w in zip(pairs, cases):
        for s in range(6):
            if s % w.sort_every == 0:
                x, y, z, pid, chi, _, _ = oracle_sort_state(prm, x, y, z, pid, chi)
            x, y, z, chi, nsub, lost, st = orc.step(prm, f_np, x, y, z, w.dt, chi, nthreads=8)
        assert np.array_equal(host(lp.id).view(np.uint64), pid) and np.array_equal(host(lp.x), x)
        assert_nsub_equal(host(lp.nsub), nsub)
        assert_chi_close(host(lp.chi), chi)
