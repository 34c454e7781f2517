"""Pins of the oracle's delete-and-fill compaction (reading C1 of DESIGN.md).

Fixed by the paper's five steps: the survivors are exactly the unflagged particles, every unflagged particle
stored below N_p - N_del stays where it is, holes below N_p - N_del are filled from the tail; two small cases
are worked by hand from the steps."""
import numpy as np
import pytest

from oracle import lp_oracle as orc


def _state(n, nb=4):
    pid = np.arange(n, dtype=np.uint64) + 100
    x = np.arange(n, dtype=np.float64) * 0.5
    chi = (np.arange(n)[:, None] * 10.0 + np.arange(nb)[None, :]).astype(np.float64)
    return x, x + 1, x + 2, pid, chi


@pytest.mark.parametrize("flags,expect", [
    # N = 8, delete {1, 5, 6}: N_del = 3, keep 5; holes below 5: {1}; fillers from {5,6,7}: {7}  => 1 <- 7
    ([0, 1, 0, 0, 0, 1, 1, 0], [0, 7, 2, 3, 4]),
    # delete {0, 2, 7}: keep 5; holes {0, 2}; fillers {5, 6}  => 0 <- 5, 2 <- 6
    ([1, 0, 1, 0, 0, 0, 0, 1], [5, 1, 6, 3, 4]),
    # only tail particles deleted: nothing moves
    ([0, 0, 0, 0, 0, 0, 1, 1], [0, 1, 2, 3, 4, 5]),
    ([0] * 8, list(range(8))),
    ([1] * 8, []),
])
def test_compact_handworked(flags, expect):
    x, y, z, pid, chi = _state(8)
    cx, cy, cz, cid, cchi = orc.compact(flags, x, y, z, pid, chi)
    e = np.array(expect, dtype=np.int64)
    assert np.array_equal(cid, pid[e]) and np.array_equal(cx, x[e]) and np.array_equal(cz, z[e])
    assert np.array_equal(cchi, chi[e])


@pytest.mark.parametrize("n,frac,seed", [(1, 0.5, 0), (2, 0.5, 1), (257, 0.3, 2), (5000, 0.05, 3), (5000, 0.9, 4)])
def test_compact_invariants(n, frac, seed):
    rng = np.random.default_rng(seed)
    flags = (rng.uniform(size=n) < frac).astype(np.int32)
    x, y, z, pid, chi = _state(n, nb=3)
    cx, cy, cz, cid, cchi = orc.compact(flags, x, y, z, pid, chi)
    keep = n - int(flags.sum())
    assert cid.shape[0] == keep
    assert set(cid.tolist()) == set(pid[flags == 0].tolist())                 # exactly the survivors, once each
    stay = np.nonzero(flags[:keep] == 0)[0]                                   # unflagged below the cut do not move
    assert np.array_equal(cid[stay], pid[stay])
    src = (cid - np.uint64(100)).astype(np.int64)                             # attributes travel together
    assert np.array_equal(cx, x[src]) and np.array_equal(cy, y[src]) and np.array_equal(cchi, chi[src])
    moved = np.nonzero(flags[:keep] == 1)[0]                                  # holes are filled from the tail, in order
    assert (src[moved] >= keep).all() and (np.diff(src[moved]) > 0).all()
