"""GPU parity of the particle exchange (lp_migrate_count / _pack / _unpack) against the
oracle's eight steps, on virtual ranks: every rank of a decomposed box is its own lp context on the one GPU,
the send buffers are handed from context to context (what NCCL or a peer copy would move).  Bit-exact:
destinations' totals, buffer contents and order, and every rank's arrays after each directional sweep."""
import itertools

import numpy as np
import pytest
import torch

import paper_2602_23434_b200 as P
from oracle import lp_oracle as orc

pytestmark = pytest.mark.gpu


def make_rank(lo, hi, n, nb, cap, rng, first_id, glo, ghi, frac_move, pingpong=False):
    lo = np.asarray(lo); hi = np.asarray(hi)
    pos = rng.uniform(lo, hi, size=(n, 3))
    pos += rng.uniform(-0.9, 0.9, size=(n, 3)) * (hi - lo) * (rng.uniform(size=(n, 1)) < frac_move)
    pos = glo + np.mod(pos - glo, ghi - glo)
    pid = (np.arange(first_id, first_id + n, dtype=np.uint64) * np.uint64(2654435761)) % np.uint64(1 << 40)
    chi = rng.uniform(size=(n, nb))
    cfg = P.make_config(8, 8, 8, (glo,) * 3, (ghi,) * 3, (1, 1, 1), cap, nb, 1.0, 1e6)
    lp = P.LP(cfg)
    pad = lambda a, shape, dt: np.concatenate([a, np.zeros(shape, dtype=dt)])
    lp.bind_particles(pad(pos[:, 0], cap - n, np.float64), pad(pos[:, 1], cap - n, np.float64),
                      pad(pos[:, 2], cap - n, np.float64), pad(pid, cap - n, np.uint64),
                      np.concatenate([chi, np.zeros((cap - n, nb))]))
    lp.set_count(n)
    if pingpong:
        lp.set_pingpong(True)
        lp.sort()                      # moves the state into the workspace twins
        torch.cuda.synchronize()
        x, y, z, i, c = lp.current()
        pos = np.stack([x[:n].cpu().numpy(), y[:n].cpu().numpy(), z[:n].cpu().numpy()], axis=1)
        pid = i[:n].cpu().numpy().view(np.uint64)
        chi = c[:n].cpu().numpy()
    return lp, (pos[:, 0].copy(), pos[:, 1].copy(), pos[:, 2].copy(), pid.copy(), chi.copy())


def decode(buf, n, nb):
    """(x, y, z, id, chi) of a send buffer laid out as arrays (include/lp.h)."""
    raw = buf.cpu().numpy()[: n * (32 + 8 * nb)]
    d = raw.view(np.float64)
    return (d[:n].copy(), d[n:2 * n].copy(), d[2 * n:3 * n].copy(), raw.view(np.uint64)[3 * n:4 * n].copy(),
            d[4 * n:].reshape(n, nb).copy())


def gpu_state(lp):
    n = lp.cfg.np
    x, y, z, i, c = lp.current()
    return (x[:n].cpu().numpy(), y[:n].cpu().numpy(), z[:n].cpu().numpy(), i[:n].cpu().numpy().view(np.uint64),
            c[:n].cpu().numpy())


@pytest.mark.parametrize("dims,nb,n_per,frac,pingpong", [
    ((2, 2, 2), 16, 3000, 0.4, False),
    ((3, 1, 2), 64, 1000 + 37, 0.7, False),
    ((2, 2, 2), 128, 500, 0.3, True),
    ((1, 2, 1), 32, 70001, 0.05, False),
])
def test_exchange_on_virtual_ranks_matches_oracle(dims, nb, n_per, frac, pingpong):
    glo, ghi = -1.0, 1.0
    rng = np.random.default_rng(11)
    faces = [np.linspace(glo, ghi, d + 1) for d in dims]
    ranks = list(itertools.product(*[range(d) for d in dims]))
    cap = 2 * n_per
    lps, ref = {}, {}
    for k, rk in enumerate(ranks):
        lo = [faces[d][rk[d]] for d in range(3)]; hi = [faces[d][rk[d] + 1] for d in range(3)]
        lps[rk], ref[rk] = make_rank(lo, hi, n_per, nb, cap, rng, k * n_per, glo, ghi, frac, pingpong)
    for axis in range(3):
        sent, packed = {}, {}
        for rk in ranks:
            lo, hi = faces[axis][rk[axis]], faces[axis][rk[axis] + 1]
            packed[rk] = orc.migrate_pack(axis, lo, hi, glo, ghi, 1, *ref[rk])
            nl, nr = lps[rk].migrate_count(axis, lo, hi)
            assert (nl, nr) == (packed[rk][2][0].shape[0], packed[rk][3][0].shape[0])
            bl, br = lps[rk].migrate_pack(nl, nr)
            sent[rk] = (bl, nl, br, nr)
            for got, want in ((decode(bl, nl, nb), packed[rk][2]), (decode(br, nr, nb), packed[rk][3])):
                for g, w in zip(got, want):
                    assert np.array_equal(g, w)
        for rk in ranks:
            def nbr(step):
                c = list(rk); c[axis] = (c[axis] + step) % dims[axis]; return tuple(c)
            if dims[axis] > 1:
                fl, nfl = sent[nbr(-1)][2], sent[nbr(-1)][3]        # the left neighbour's right buffer
                fr, nfr = sent[nbr(+1)][0], sent[nbr(+1)][1]
                ofl, ofr = packed[nbr(-1)][3], packed[nbr(+1)][2]
            else:
                fl = fr = None; nfl = nfr = 0; ofl = ofr = None
            ref[rk] = orc.migrate_unpack(packed[rk][1], ofl, ofr, *ref[rk])
            n_new = lps[rk].migrate_unpack(fl, nfl, fr, nfr)
            assert n_new == ref[rk][0].shape[0]
        torch.cuda.synchronize()
        for rk in ranks:
            for g, w in zip(gpu_state(lps[rk]), ref[rk]):
                assert np.array_equal(g, w)
    # everybody at home
    for rk in ranks:
        x, y, z, _, _ = gpu_state(lps[rk])
        for d, a in enumerate((x, y, z)):
            assert (a >= faces[d][rk[d]]).all() and (a < faces[d][rk[d] + 1]).all()


def test_exchange_state_errors_and_capacity():
    rng = np.random.default_rng(3)
    lp, st = make_rank([-1, -1, -1], [0, 1, 1], 100, 16, 120, rng, 0, -1.0, 1.0, 0.5)
    B = P.binding
    with pytest.raises(B.LPError) as e:
        lp.migrate_pack(0, 0)
    assert e.value.status == B.LP_ERR_STATE
    nl, nr = lp.migrate_count(0, -1.0, 0.0)
    with pytest.raises(B.LPError) as e:
        lp.migrate_unpack(None, 0, None, 0)
    assert e.value.status == B.LP_ERR_STATE
    bl, br = lp.migrate_pack(nl, nr)
    big = lp.migrate_buffer(200)
    with pytest.raises(B.LPError) as e:                 # more arrivals than the arrays can take
        lp.migrate_unpack(big, 200, None, 0)
    assert e.value.status == B.LP_ERR_WORKSPACE
    n = lp.migrate_unpack(None, 0, None, 0)             # nobody arrives: the holes are compacted away
    assert n == 100 - nl - nr
    want = orc.migrate_unpack(orc.migrate_pack(0, -1.0, 0.0, -1.0, 1.0, 1, *st)[1], None, None, *st)
    torch.cuda.synchronize()
    for g, w in zip(gpu_state(lp), want):
        assert np.array_equal(g, w)
    lp.sort()                                           # a sort invalidates a count
    nl, nr = lp.migrate_count(0, -1.0, 0.0)
    lp.sort()
    with pytest.raises(B.LPError):
        lp.migrate_pack(nl, nr)


@pytest.mark.parametrize("n,lo,hi", [(0, -1.0, 0.0), (1, 0.5, 1.0), (1, -1.0, 1.0), (37, 0.999, 1.0), (4097, -1.0, 1.0)])
def test_exchange_degenerate_sets(n, lo, hi):
    """No particles, one particle, (almost) everybody leaving, nobody leaving: counts, buffers and the state after
    an exchange in which nothing arrives follow the oracle."""
    rng = np.random.default_rng(n)
    nb, cap = 16, max(n, 1)
    cfg = P.make_config(4, 4, 4, (-1.0,) * 3, (1.0,) * 3, (1, 1, 1), cap, nb, 1.0, 1e6)
    lp = P.LP(cfg)
    pos = rng.uniform(-1, 0.99, size=(cap, 3)); pid = np.arange(cap, dtype=np.uint64) + np.uint64(7)
    chi = rng.uniform(size=(cap, nb))
    lp.bind_particles(pos[:, 0], pos[:, 1], pos[:, 2], pid, chi)
    lp.set_count(n)
    st = tuple(a[:n].copy() for a in (pos[:, 0], pos[:, 1], pos[:, 2], pid, chi))
    dest, holes, left, right = orc.migrate_pack(0, lo, hi, -1.0, 1.0, 1, *st)
    nl, nr = lp.migrate_count(0, lo, hi)
    assert (nl, nr) == (left[0].shape[0], right[0].shape[0])
    bl, br = lp.migrate_pack(nl, nr)
    for got, want in ((decode(bl, nl, nb), left), (decode(br, nr, nb), right)):
        for g, w_ in zip(got, want):
            assert np.array_equal(g, w_)
    n_new = lp.migrate_unpack(None, 0, None, 0)
    want = orc.migrate_unpack(holes, None, None, *st)
    assert n_new == want[0].shape[0] == n - nl - nr
    torch.cuda.synchronize()
    for g, w_ in zip(gpu_state(lp), want):
        assert np.array_equal(g, w_)
    if nl + nr:                                             # everything that left comes back in: the count is restored
        assert lp.migrate_count(0, -1.0, 1.0) == (0, 0)
        lp.migrate_pack(0, 0)
        assert lp.migrate_unpack(bl, nl, br, nr) == n
        back = orc.migrate_unpack(np.zeros(0, dtype=np.int64), left, right, *want)
        for g, w_ in zip(gpu_state(lp), back):
            assert np.array_equal(g, w_)


def test_diag_between_count_and_pack_leaves_the_exchange_alone():
    """lp.h allows any call that moves no particle between lp_migrate_count and lp_migrate_pack.  lp_get_diag is
    one, and its per-block partial sums used to land on the device copy of the leaver totals that the pack kernel
    read (round-2 advisor finding): count -> diag -> pack -> unpack must give the oracle's buffers and state."""
    rng = np.random.default_rng(17)
    nb = 32
    lp, st = make_rank([-1, -1, -1], [0, 1, 1], 3000 + 11, nb, 3200, rng, 5, -1.0, 1.0, 0.5)
    dest, holes, left, right = orc.migrate_pack(0, -1.0, 0.0, -1.0, 1.0, 1, *st)
    nl, nr = lp.migrate_count(0, -1.0, 0.0)
    assert (nl, nr) == (left[0].shape[0], right[0].shape[0]) and nl > 0 and nr > 0
    d = lp.diag()                                           # writes fp64 partial sums into the shared scratch
    assert d["np"] == 3000 + 11 and d["number"] > 0
    bl, br = lp.migrate_pack(nl, nr)
    torch.cuda.synchronize()
    for got, want in ((decode(bl, nl, nb), left), (decode(br, nr, nb), right)):
        for g, w_ in zip(got, want):
            assert np.array_equal(g, w_)
    lp.diag()
    n_new = lp.migrate_unpack(br, nr, bl, nl)               # the leavers come back in, right buffer first
    want = orc.migrate_unpack(holes, right, left, *st)
    assert n_new == want[0].shape[0] == 3000 + 11
    torch.cuda.synchronize()
    for g, w_ in zip(gpu_state(lp), want):
        assert np.array_equal(g, w_)
