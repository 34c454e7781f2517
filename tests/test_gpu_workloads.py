"""GPU parity on the five BASELINE.json workloads.

Workloads 1-2 run in full on both sides.  Workloads 3-5 run at full size on the GPU in the launch
configuration bench.py times; the oracle recomputes a seeded SAMPLE of particles one by one (each
particle's step depends only on its own state and the fields), and properties that hold at any
size (sort order, id permutation, number conservation, positions in the box) cover the rest."""
import math

import numpy as np
import pytest
import torch

import lp_inputs as I
import paper_2602_23434_b200 as P
from oracle import lp_oracle as orc

from lp_testlib import (REL_TOL, assert_chi_close, assert_nsub_equal, fields_to_numpy, oracle_params,
                        u_rad_of, workload1_dt)

pytestmark = pytest.mark.gpu


def host(t):
    return t.detach().cpu().numpy()


def test_workload1_synchrotron_full_and_analytic():
    """16^3, 1024 particles, 64 bins, 100 steps, dt from the loss CFL; also against the analytic
    cooled power law (first-order accurate scheme, same bound as the oracle pin)."""
    w = I.workload(1)
    dt = workload1_dt(w)
    fields = I.make_fields(w)
    f_np = fields_to_numpy(fields)
    x, y, z, pid = I.make_particles(w)
    chi = I.make_spectrum(w, jitter=False)
    lp = P.LP(P.config_from_workload(w))
    lp.set_fields(fields); lp.bind_particles(x, y, z, pid, chi); lp.bind_diag()
    prm = oracle_params(w, 0.0)
    for _ in range(w.steps):
        lp.step(dt)
        x, y, z, chi, nsub, lost, st = orc.step(prm, f_np, x, y, z, dt, chi, nthreads=8)
    torch.cuda.synchronize()
    assert (nsub == 1).all()
    assert_nsub_equal(host(lp.nsub), nsub)
    assert np.array_equal(host(lp.x), x)              # v = 0: nobody moves
    g = host(lp.chi)
    assert_chi_close(g, chi)
    # analytic: exact bin contents of the cooled power law (number conserved along eps0/(1+c eps0 t))
    E, dE, Ec = orc.bin_table(w.nbins, w.e_min, w.e_max)
    ea, eb = w.support; p = w.p_index
    cr = 0.5 * w.b0 ** 2; t = w.steps * dt
    K = (1 - p) / (eb ** (1 - p) - ea ** (1 - p))
    with np.errstate(divide="ignore", invalid="ignore"):
        e0 = np.where(cr * E * t < 1.0, E / (1.0 - cr * E * t), np.inf)
    cum = K * (np.clip(e0, ea, eb) ** (1 - p) - ea ** (1 - p)) / (1 - p)
    exact = cum[1:] - cum[:-1]
    cutoff = eb / (1 + cr * eb * t)
    smooth = (E[:-1] > 2e2) & (E[1:] < 0.5 * cutoff)
    assert smooth.sum() > 10
    assert np.max(np.abs(g[0][smooth] * dE[smooth] / exact[smooth] - 1)) < 0.04


def test_workload2_adiabatic_staged_full():
    """64^3 clamped, 65,536 particles, 128 bins, 200 steps of the staged API with the homologous
    fields advanced between the stages; checked against the oracle and E ~ rho^(1/3)."""
    w = I.workload(2)
    dt = w.dt
    x, y, z, pid = I.make_particles(w)
    chi = I.make_spectrum(w, jitter=True)
    chi0 = chi.copy()
    lp = P.LP(P.config_from_workload(w))
    lp.bind_particles(x, y, z, pid, chi); lp.bind_diag()
    prm = oracle_params(w, 0.0)
    x0 = x.copy()
    for s in range(w.steps):
        f0 = I.make_fields(w, t=s * dt); f1 = I.make_fields(w, t=(s + 1) * dt)
        lp.set_fields(f0); lp.push(dt, 0)
        lp.set_fields(f1); lp.push(dt, 1); lp.spectral_update(dt)
        n0, n1 = fields_to_numpy(f0), fields_to_numpy(f1)
        k1, rho_old, xs = orc.push_stage0(prm, n0, x, y, z, dt, nthreads=8)
        x, y, z, st = orc.push_stage1(prm, n1, x, y, z, xs, k1, dt, nthreads=8)
        chi, nsub, lost = orc.spectral_update(prm, n1, x, y, z, rho_old, dt, chi, nthreads=8)
    torch.cuda.synchronize()
    assert np.array_equal(host(lp.x), x) and np.array_equal(host(lp.y), y) and np.array_equal(host(lp.z), z)
    assert_nsub_equal(host(lp.nsub), nsub)
    g = host(lp.chi)
    assert_chi_close(g, chi)
    t_end = w.steps * dt
    assert np.max(np.abs(x - x0 * (1 + w.alpha * t_end))) < 1e-12        # Heun exact for this flow
    ratio = (g / chi0)[:, w.nbins // 4: w.nbins // 2]
    expect = ((1 + w.alpha * t_end) ** -3) ** ((w.p_index - 1) / 3)
    assert np.max(np.abs(ratio / expect - 1)) < 0.12                      # first order in 128 bins


_FIELD_CACHE = {}


def cached_fields(w, dev):
    """Fields depend on the grid and the seed only, not on the bin count: reuse across the sweep."""
    k = (w.index, w.n, w.seed)
    if k not in _FIELD_CACHE:
        _FIELD_CACHE.clear()                      # keep at most one grid resident
        f = I.make_fields(w, device=dev)
        _FIELD_CACHE[k] = (f, fields_to_numpy(f))
    return _FIELD_CACHE[k]


def run_sampled(w, steps, nsample=2048, check_sort=True, diag="full", pingpong=False):
    """Run `steps` lp_step on the GPU at full size and the oracle on a sample; compare by id.
    diag = "nsub": only n_sub is bound, so the DIAG=false kernel instantiations run -- the ones bench.py
    times (it binds no `lost` output); the number-conservation property needs `lost` and is then skipped."""
    dev = "cuda"
    fields, f_np = cached_fields(w, dev)
    u_rad = u_rad_of(w, fields)
    x, y, z, pid = I.make_particles(w, shuffle_ids=True)
    chi_dev = torch.from_numpy(I.make_spectrum(w.scaled(np=1), jitter=False)).to(dev)
    rng = np.random.Generator(np.random.PCG64(w.seed + 2000))
    amp = 1.0 + 0.5 * rng.uniform(size=w.np)
    chi_dev = (torch.from_numpy(amp).to(dev)[:, None] * chi_dev).contiguous()     # [np, nbins]
    lp = P.LP(P.config_from_workload(w, u_rad=u_rad))
    lp.set_fields(fields)
    lp.bind_particles(x, y, z, pid, chi_dev)
    lp.bind_diag(nsub=True, lost=(diag == "full"))
    lp.set_pingpong(pingpong)
    n0 = lp.diag()["number"]
    # oracle sample (ids chosen by a seeded draw)
    srng = np.random.default_rng(12345)
    sel = np.sort(srng.choice(w.np, size=min(nsample, w.np), replace=False))
    prm = oracle_params(w, u_rad)
    sx, sy, sz, sid = x[sel].copy(), y[sel].copy(), z[sel].copy(), pid[sel].copy()
    schi = host(chi_dev[torch.from_numpy(sel).to(dev)])
    lost_total = 0.0
    for s in range(steps):
        lp.step(w.dt)
        sx, sy, sz, schi, snsub, slost, st = orc.step(prm, f_np, sx, sy, sz, w.dt, schi, nthreads=8)
        if diag == "full":
            lost_total += lp.diag()["lost"]
    torch.cuda.synchronize()
    gid = host(lp.id).view(np.uint64)
    # properties at full size
    assert np.array_equal(np.sort(gid), np.arange(w.np, dtype=np.uint64))          # a permutation of the ids
    gx, gy, gz = host(lp.x), host(lp.y), host(lp.z)
    for a in (gx, gy, gz):
        assert (a >= -1.0).all() and (a < 1.0).all()
    d = lp.diag()
    if diag == "full":
        assert abs((d["number"] + lost_total) / n0 - 1) < 1e-11
    assert d["n_capped"] == 0 and d["n_outside"] == 0
    if check_sort and w.sort_every:
        assert d["sorts"] == (steps + w.sort_every - 1) // w.sort_every
    # sampled particles, matched by id
    where = np.empty(w.np, dtype=np.int64); where[gid.astype(np.int64)] = np.arange(w.np)
    loc = where[sid.astype(np.int64)]
    assert np.array_equal(gx[loc], sx) and np.array_equal(gy[loc], sy) and np.array_equal(gz[loc], sz)
    assert_nsub_equal(host(lp.nsub)[loc], snsub)
    gchi = host(lp.chi[torch.from_numpy(loc).to(dev)])
    assert_chi_close(gchi, schi)
    return lp, d, snsub


def test_workload3_turbulent_sampled():
    w = I.workload(3)
    lp, d, nsub = run_sampled(w, steps=5)
    assert d["max_substeps"] >= 1


def test_workload3_full_length_bench_kernels():
    """All 50 steps of BASELINE.json configs[2] in the kernels bench.py times (no `lost` output bound)."""
    w = I.workload(3)
    assert w.steps == 50
    lp, d, nsub = run_sampled(w, steps=w.steps, diag="nsub", pingpong=True)
    assert d["steps"] == 50


def check_sorted_after_explicit_sort(lp):
    lp.sort()
    _, key = lp.interpolate(want_fields=False)
    key = host(key).view(np.uint32).astype(np.int64)
    gid = host(lp.id).view(np.uint64)
    dk = np.diff(key)
    assert (dk >= 0).all()
    same = dk == 0
    assert (np.diff(gid.astype(np.int64))[same] > 0).all()


def test_workload4_large_sampled_with_resort():
    """16.7M particles, 256^3, 64 bins, sort_every = 10: 11 steps so that two sorts happen; after the
    second sort + one step the order is still (key, id) ascending up to the drift of that step, so
    the order property is checked right after an explicit lp_sort."""
    w = I.workload(4)
    lp, d, nsub = run_sampled(w, steps=11, nsample=4096)
    assert d["sorts"] == 2
    check_sorted_after_explicit_sort(lp)


def test_workload4_full_length_bench_kernels():
    """All 20 steps of BASELINE.json configs[3] (two re-sorts) in the kernels bench.py times."""
    w = I.workload(4)
    assert w.steps == 20
    lp, d, nsub = run_sampled(w, steps=w.steps, nsample=4096, diag="nsub", pingpong=True)     # as bench.py runs it
    assert d["sorts"] == 2 and d["steps"] == 20
    check_sorted_after_explicit_sort(lp)


@pytest.mark.parametrize("nbins", [16, 32, 64, 128, 256, 512])
def test_workload5_bin_sweep_sampled(nbins):
    w = I.workload(5).scaled(nbins=nbins)
    lp, d, nsub = run_sampled(w, steps=2, nsample=1024)
    expected_typical = {16: 1, 32: 1, 64: 1, 128: 2, 256: 5, 512: 10}[nbins]
    assert 0.4 * expected_typical <= np.median(np.abs(nsub)) <= 2.5 * expected_typical


@pytest.mark.parametrize("nbins", [16, 32, 64, 128, 256, 512])
def test_workload5_full_length_bench_kernels(nbins):
    """All 10 steps of BASELINE.json configs[4] at every bin count, in the kernels bench.py times."""
    w = I.workload(5).scaled(nbins=nbins)
    assert w.steps == 10
    lp, d, nsub = run_sampled(w, steps=w.steps, nsample=1024, diag="nsub", pingpong=True)
    assert d["steps"] == 10 and d["sorts"] == 1
