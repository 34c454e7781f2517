"""Pins of the oracle's particle exchange (readings M1-M3 of DESIGN.md section 3).

Fixed by the paper's steps and by what an exchange must achieve: a hand-worked two-rank case
(tests/golden/migrate_handworked.txt), the destination rule against the owner found by brute force, and on
a 3 x 2 x 2 decomposition after the three directional sweeps: every particle sits on the rank that owns its
position, no particle is lost or duplicated, all parameters travel together, particles that stay keep their
slot unless they are tail fillers."""
import itertools

import numpy as np
import pytest

from oracle import lp_oracle as orc


def _state(x, pid, nb=3):
    x = np.asarray(x, dtype=np.float64)
    pid = np.asarray(pid, dtype=np.uint64)
    chi = pid.astype(np.float64)[:, None] * 100.0 + np.arange(nb)[None, :]
    return x, x * 0.0 + 0.25, x * 0.0 + 0.75, pid, chi


def test_two_rank_exchange_handworked(golden):
    g = golden("migrate_handworked.txt")
    ranks = []
    for r, (lo, hi) in enumerate([(0.0, 4.0), (4.0, 8.0)]):
        st = _state(g["r%d_x" % r], [int(v) for v in g["r%d_id" % r]])
        dest, holes, left, right = orc.migrate_pack(0, lo, hi, 0.0, 8.0, 1, *st)
        assert dest.tolist() == [int(v) for v in g["r%d_dest" % r]]
        assert holes.tolist() == [int(v) for v in g["r%d_holes" % r]]
        assert left[3].tolist() == [int(v) for v in g["r%d_left_ids" % r]]
        assert right[3].tolist() == [int(v) for v in g["r%d_right_ids" % r]]
        ranks.append((st, holes, left, right))
    for r in range(2):
        st, holes, _, _ = ranks[r]
        other = ranks[1 - r]
        # from my left neighbour comes what it sent to its right, and the other way round
        x, y, z, pid, chi = orc.migrate_unpack(holes, other[3], other[2], *st)
        assert pid.tolist() == [int(v) for v in g["r%d_after_ids" % r]]
        assert np.array_equal(chi[:, 0], pid.astype(np.float64) * 100.0)      # rows travelled with their ids
        assert np.array_equal(y, np.full(pid.shape[0], 0.25))


@pytest.mark.parametrize("periodic", [1, 0])
def test_destination_is_the_owner_found_by_brute_force(periodic):
    """P equal slabs of a box; a particle that moved by less than a slab width belongs to the slab found by
    searching the faces, which must be the rank itself (0), its left (1) or its right (2) neighbour."""
    rng = np.random.default_rng(5)
    P, glo, ghi = 5, -1.0, 1.0
    faces = np.linspace(glo, ghi, P + 1)
    w = faces[1] - faces[0]
    for me in range(P):
        x0 = rng.uniform(faces[me], faces[me + 1], size=400)
        x = x0 + rng.uniform(-0.99 * w, 0.99 * w, size=400)
        if periodic:
            x = glo + np.mod(x - glo, ghi - glo)
        else:
            keep = (x >= glo) & (x < ghi)
            x = x[keep]
        for xv in x:
            owner = max(k for k in range(P) if faces[k] <= xv)               # brute force over the faces
            want = 0 if owner == me else (1 if owner == (me - 1) % P else 2)
            assert owner in (me, (me - 1) % P, (me + 1) % P)
            assert orc.migrate_dest(xv, faces[me], faces[me + 1], glo, ghi, periodic) == want


def test_face_belongs_to_the_upper_rank_and_single_rank_keeps_everything():
    assert orc.migrate_dest(4.0, 0.0, 4.0, 0.0, 8.0, 1) == 2          # x == hi leaves to the right
    assert orc.migrate_dest(4.0, 4.0, 8.0, 0.0, 8.0, 1) == 0          # x == lo stays
    x = np.random.default_rng(1).uniform(-1, 1, size=100)
    for xv in x:                                                      # one rank on the axis: nobody leaves
        assert orc.migrate_dest(xv, -1.0, 1.0, -1.0, 1.0, 1) == 0


def _decomp(dims, glo, ghi):
    faces = [np.linspace(glo, ghi, d + 1) for d in dims]
    ranks = list(itertools.product(*[range(d) for d in dims]))
    return faces, ranks


def run_exchange(dims, state_by_rank, glo, ghi, periodic=1):
    """The three directional sweeps over all ranks of a dims[0] x dims[1] x dims[2] decomposition."""
    faces, ranks = _decomp(dims, glo, ghi)
    for axis in range(3):
        packed = {}
        for rk in ranks:
            lo, hi = faces[axis][rk[axis]], faces[axis][rk[axis] + 1]
            packed[rk] = orc.migrate_pack(axis, lo, hi, glo, ghi, periodic, *state_by_rank[rk])
        for rk in ranks:
            def nb(step):
                c = list(rk); c[axis] = (c[axis] + step) % dims[axis]; return tuple(c)
            from_left = packed[nb(-1)][3] if dims[axis] > 1 else None          # the left neighbour's right buffer
            from_right = packed[nb(+1)][2] if dims[axis] > 1 else None
            state_by_rank[rk] = orc.migrate_unpack(packed[rk][1], from_left, from_right, *state_by_rank[rk])
    return state_by_rank


@pytest.mark.parametrize("seed", [0, 1, 2])
def test_three_sweeps_bring_every_particle_to_its_owner(seed):
    rng = np.random.default_rng(seed)
    dims, glo, ghi, nb = (3, 2, 2), -1.0, 1.0, 4
    faces, ranks = _decomp(dims, glo, ghi)
    n_per = 300
    state, before, next_id = {}, {}, 0
    for rk in ranks:
        lo = np.array([faces[d][rk[d]] for d in range(3)]); hi = np.array([faces[d][rk[d] + 1] for d in range(3)])
        pos = rng.uniform(lo, hi, size=(n_per, 3))
        pos += rng.uniform(-0.9, 0.9, size=(n_per, 3)) * (hi - lo) * (rng.uniform(size=(n_per, 1)) < 0.4)
        pos = glo + np.mod(pos - glo, ghi - glo)                     # Particles_Boundary: wrapped into the box
        pid = np.arange(next_id, next_id + n_per, dtype=np.uint64); next_id += n_per
        chi = rng.uniform(size=(n_per, nb))
        state[rk] = (pos[:, 0].copy(), pos[:, 1].copy(), pos[:, 2].copy(), pid, chi)
        for k in range(n_per):
            before[int(pid[k])] = (pos[k].copy(), chi[k].copy())
    start = {rk: tuple(a.copy() for a in state[rk]) for rk in ranks}
    state = run_exchange(dims, state, glo, ghi)
    seen = []
    for rk in ranks:
        x, y, z, pid, chi = state[rk]
        pos = np.stack([x, y, z], axis=1)
        for d in range(3):                                           # everybody is at home
            assert (pos[:, d] >= faces[d][rk[d]]).all() and (pos[:, d] < faces[d][rk[d] + 1]).all()
        for k in range(pid.shape[0]):                                # parameters travelled together, unchanged
            p0, c0 = before[int(pid[k])]
            assert np.array_equal(pos[k], p0) and np.array_equal(chi[k], c0)
        seen += pid.tolist()
        # a particle that was at home from the start and whose slot survives every sweep has not moved
        sx, sy, sz, sid, _ = start[rk]
        n_min = min(pid.shape[0], sid.shape[0])
        home = np.ones(sid.shape[0], dtype=bool)
        for d, s in enumerate((sx, sy, sz)):
            home &= (s >= faces[d][rk[d]]) & (s < faces[d][rk[d] + 1])
        stay = np.nonzero(home[:n_min] & (pid[:n_min] == sid[:n_min]))[0]
        assert stay.size > 0.3 * n_per
    assert sorted(seen) == list(range(next_id))                      # nobody lost, nobody twice


def test_more_arrivals_than_holes_and_fewer():
    # rank with 4 particles, 1 leaver, 3 arrivals: one hole filled, two appended, in buffer order
    st = _state([0.5, 1.5, 9.0, 2.5], [1, 2, 3, 4])
    dest, holes, left, right = orc.migrate_pack(0, 0.0, 4.0, 0.0, 16.0, 1, *st)
    assert holes.tolist() == [2] and right[3].tolist() == [3]
    arr_l = _state([1.0, 1.1], [50, 51]); arr_r = _state([3.0], [60])
    x, y, z, pid, chi = orc.migrate_unpack(holes, arr_l, arr_r, *st)
    assert pid.tolist() == [1, 2, 50, 4, 51, 60]
    # 3 leavers, 1 arrival: holes 0 2 3 -> 0 <- 70; holes 2, 3 compacted: keep = 3, hole below 3: {2}, filler {4}
    st = _state([9.0, 1.5, 9.5, 10.0, 2.5], [1, 2, 3, 4, 5])
    dest, holes, left, right = orc.migrate_pack(0, 0.0, 4.0, 0.0, 16.0, 1, *st)
    assert holes.tolist() == [0, 2, 3]
    x, y, z, pid, chi = orc.migrate_unpack(holes, _state([0.1], [70]), None, *st)
    assert pid.tolist() == [70, 2, 5]
