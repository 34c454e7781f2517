"""GPU tests of the chunked growth of the particle storage (lp_rebind, LP.reserve / LP.shrink; PAPER.md:176-184
Listing 1, Reserve() / Shrink() of Listing 2): particles are injected past the capacity the context was created
with, deleted again, trailing chunks released -- the state must follow the oracle through all of it."""
import numpy as np
import pytest
import torch

import lp_inputs as I
import paper_2602_23434_b200 as P
from oracle import lp_oracle as orc
from lp_testlib import assert_chi_close, assert_nsub_equal, fields_to_numpy, oracle_params, u_rad_of

pytestmark = pytest.mark.gpu
B = P.binding


def host(t):
    return t.detach().cpu().numpy()


def oracle_step(prm, f_np, st, dt, sort):
    x, y, z, pid, chi = st
    if sort:
        perm = orc.sort_perm(orc.cell_key(prm, x, y, z), pid)
        x, y, z, pid, chi = x[perm], y[perm], z[perm], pid[perm], chi[perm]
    x, y, z, chi, nsub, lost, status = orc.step(prm, f_np, x, y, z, dt, chi, nthreads=8)
    return [x, y, z, pid, chi], nsub


def check(lp, st, nsub=None):
    n = st[0].shape[0]
    assert lp.cfg.np == n and lp.diag()["np"] == n
    assert np.array_equal(host(lp.id)[:n].view(np.uint64), st[3])
    for g, w in zip((lp.x, lp.y, lp.z), st[:3]):
        assert np.array_equal(host(g)[:n], w)
    assert_chi_close(host(lp.chi)[:n], st[4])
    if nsub is not None:
        assert_nsub_equal(host(lp.nsub)[:n], nsub)


@pytest.mark.parametrize("pingpong", [False, True])
@pytest.mark.parametrize("nbins", [64, 512])
def test_reserve_past_the_create_time_capacity_then_shrink(nbins, pingpong):
    e = 10
    n0, n_add = 5000, 3000
    cap0 = B.lp_chunked_capacity(n0, e)
    assert cap0 == 5120
    w = I.workload(3).scaled(n=12, np=cap0, nbins=nbins, sort_every=1)
    fields = I.make_fields(w, device="cpu")
    u_rad = u_rad_of(w, fields)
    f_np = fields_to_numpy(fields)
    prm = oracle_params(w, u_rad)
    x, y, z, pid = I.make_particles(w, shuffle_ids=True)
    chi = I.make_spectrum(w)
    lp = P.LP(P.config_from_workload(w, u_rad=u_rad))
    lp.set_fields(fields)
    lp.bind_particles(x, y, z, pid, chi)
    lp.bind_diag(nsub=True, lost=False)
    lp.set_pingpong(pingpong)
    lp.set_count(n0)
    st = [a[:n0].copy() for a in (x, y, z, pid, chi)]
    for _ in range(2):
        lp.step(w.dt)
        st, nsub = oracle_step(prm, f_np, st, w.dt, True)
    check(lp, st, nsub)

    # Reserve(): 8000 particles need 8 chunks of 1024
    assert lp.reserve(100, e) == cap0                       # still fits: nothing happens
    ws_before = lp.workspace.data_ptr()
    assert lp.reserve(n_add, e) == 8192 and B.lp_capacity(lp.ctx) == 8192
    assert lp.workspace.data_ptr() != ws_before
    check(lp, st)                                           # the state moved along, fields still set
    rng = np.random.default_rng(77)
    add = [rng.uniform(-1, 1, size=n_add) for _ in range(3)]
    add_id = np.arange(1 << 36, (1 << 36) + n_add, dtype=np.uint64)          # wider ids than any so far
    add_chi = I.make_spectrum(w.scaled(np=n_add, seed=w.seed + 5))
    cx, cy, cz, cid, cchi = lp.current()
    for t, a in zip((cx, cy, cz), add):
        t[n0:n0 + n_add] = torch.from_numpy(a).to(t.device)
    cid[n0:n0 + n_add] = torch.from_numpy(add_id.view(np.int64)).to(cid.device)
    cchi[n0:n0 + n_add] = torch.from_numpy(add_chi).to(cchi.device)
    lp.set_count(n0 + n_add)
    st = [np.concatenate([s, a]) for s, a in zip(st, add + [add_id, add_chi])]
    for _ in range(2):
        lp.step(w.dt)
        st, nsub = oracle_step(prm, f_np, st, w.dt, True)
    check(lp, st, nsub)

    # delete three quarters, Shrink(): 2000 particles fit 2 chunks
    flag = (rng.uniform(size=n0 + n_add) < 0.75).astype(np.int32)
    n_new = lp.compact(torch.from_numpy(flag).to(lp.device))
    st = list(orc.compact(flag, *st))
    assert n_new == st[0].shape[0]
    want_cap = B.lp_chunked_capacity(n_new, e)
    assert lp.shrink(e) == want_cap < 8192
    check(lp, st)
    lp.step(w.dt)
    st, nsub = oracle_step(prm, f_np, st, w.dt, True)
    check(lp, st, nsub)
    with pytest.raises(B.LPError):                           # capacity below the count is refused
        B.lp_rebind(lp.ctx, n_new - 1, lp.workspace.data_ptr(), lp.workspace_bytes, *[t.data_ptr() for t in lp.current()], None)


def test_exchange_arrivals_beyond_capacity_grow_the_arrays():
    """Step 6 of the exchange: the container is resized between pack and unpack."""
    rng = np.random.default_rng(5)
    n, nb = 1000, 32
    cfg = P.make_config(8, 8, 8, (-1.0,) * 3, (1.0,) * 3, (1, 1, 1), n, nb, 1.0, 1e6)
    lp = P.LP(cfg)
    pos = rng.uniform(-1, 1, size=(n, 3)); pos[:, 0] = rng.uniform(-1, 0.1, size=n)      # a few beyond hi = 0
    pid = np.arange(n, dtype=np.uint64); chi = rng.uniform(size=(n, nb))
    lp.bind_particles(pos[:, 0], pos[:, 1], pos[:, 2], pid, chi)
    st = (pos[:, 0].copy(), pos[:, 1].copy(), pos[:, 2].copy(), pid, chi)
    nl, nr = lp.migrate_count(0, -1.0, 0.0)
    bl, br = lp.migrate_pack(nl, nr)
    dest, holes, left, right = orc.migrate_pack(0, -1.0, 0.0, -1.0, 1.0, 1, *st)
    n_in = nl + nr + 500                                       # 500 more arrivals than holes
    arr = (rng.uniform(-1, 0, size=n_in), rng.uniform(-1, 1, size=n_in), rng.uniform(-1, 1, size=n_in),
           np.arange(5000, 5000 + n_in, dtype=np.uint64), rng.uniform(size=(n_in, nb)))
    raw = np.zeros(n_in * (32 + 8 * nb), dtype=np.uint8)
    d = raw.view(np.float64)
    d[:n_in], d[n_in:2 * n_in], d[2 * n_in:3 * n_in] = arr[0], arr[1], arr[2]
    raw.view(np.uint64)[3 * n_in:4 * n_in] = arr[3]
    d[4 * n_in:] = arr[4].reshape(-1)
    buf = torch.from_numpy(raw).to(lp.device)
    with pytest.raises(B.LPError) as err:
        lp.migrate_unpack(buf, n_in, None, 0)
    assert err.value.status == B.LP_ERR_WORKSPACE
    lp.reserve(500, e=8)
    assert lp.capacity == B.lp_chunked_capacity(n + 500, 8)
    n_new = lp.migrate_unpack(buf, n_in, None, 0)
    want = orc.migrate_unpack(holes, arr, None, *st)
    assert n_new == want[0].shape[0] == n + 500
    torch.cuda.synchronize()
    x, y, z, i, c = lp.current()
    got = (host(x)[:n_new], host(y)[:n_new], host(z)[:n_new], host(i)[:n_new].view(np.uint64), host(c)[:n_new])
    for g, w_ in zip(got, want):
        assert np.array_equal(g, w_)
