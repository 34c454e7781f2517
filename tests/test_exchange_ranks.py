"""Host logic of the multi-rank particle exchange (paper_2602_23434_b200/exchange.py) on CPU:
gloo ranks, each with a stand-in for `LP` whose migrate_* calls run the ORACLE on CPU tensors in the library's
buffer layout.  What is tested is the plumbing: who sends what to whom, count exchange, buffer sizing, the
left / right pairing when both neighbours are the same rank.  (The kernels themselves are compared with the
oracle on the GPU, tests/test_gpu_migrate.py.)"""
import itertools
import os
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

GLO, GHI, NB = -1.0, 1.0, 4


class OracleLP:
    """migrate_count / migrate_buffer / migrate_pack / migrate_unpack of LP, on the CPU through the oracle."""

    def __init__(self, state):
        self.state = state
        self._packed = None

    def migrate_buffer(self, n):
        return torch.zeros(max(1, n) * (32 + 8 * NB), dtype=torch.uint8)

    def migrate_count(self, axis, lo, hi):
        from oracle import lp_oracle as orc
        self._packed = orc.migrate_pack(axis, lo, hi, GLO, GHI, 1, *self.state)
        return self._packed[2][0].shape[0], self._packed[3][0].shape[0]

    @staticmethod
    def _encode(b):
        n = b[0].shape[0]
        raw = np.zeros(max(1, n) * (32 + 8 * NB), dtype=np.uint8)
        d = raw.view(np.float64)
        d[:n], d[n:2 * n], d[2 * n:3 * n] = b[0], b[1], b[2]
        raw.view(np.uint64)[3 * n:4 * n] = b[3]
        d[4 * n:4 * n + n * NB] = b[4].reshape(-1)
        return torch.from_numpy(raw)

    @staticmethod
    def _decode(t, n):
        raw = t.numpy()
        d = raw.view(np.float64)
        return (d[:n].copy(), d[n:2 * n].copy(), d[2 * n:3 * n].copy(), raw.view(np.uint64)[3 * n:4 * n].copy(),
                d[4 * n:4 * n + n * NB].reshape(n, NB).copy())

    def migrate_pack(self, n_left, n_right):
        return self._encode(self._packed[2]), self._encode(self._packed[3])

    def migrate_unpack(self, from_left, n_from_left, from_right, n_from_right):
        from oracle import lp_oracle as orc
        self.state = orc.migrate_unpack(self._packed[1], self._decode(from_left, n_from_left),
                                        self._decode(from_right, n_from_right), *self.state)
        return self.state[0].shape[0]


def initial_state(rank_coord, dims, n_per):
    faces = [np.linspace(GLO, GHI, d + 1) for d in dims]
    flat = int(np.ravel_multi_index(rank_coord, dims))
    rng = np.random.default_rng(100 + flat)
    lo = np.array([faces[d][rank_coord[d]] for d in range(3)]); hi = np.array([faces[d][rank_coord[d] + 1] for d in range(3)])
    pos = rng.uniform(lo, hi, size=(n_per, 3))
    pos += rng.uniform(-0.9, 0.9, size=(n_per, 3)) * (hi - lo) * (rng.uniform(size=(n_per, 1)) < 0.5)
    pos = GLO + np.mod(pos - GLO, GHI - GLO)
    pid = np.arange(flat * n_per, (flat + 1) * n_per, dtype=np.uint64)
    chi = pid.astype(np.float64)[:, None] + 0.125 * np.arange(NB)[None, :]
    return (pos[:, 0].copy(), pos[:, 1].copy(), pos[:, 2].copy(), pid, chi), lo, hi


def _rank_main(rank, dims, n_per, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    world = int(np.prod(dims))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_2602_23434_b200 import exchange as X
    coord = tuple(int(c) for c in np.unravel_index(rank, dims))
    state, lo, hi = initial_state(coord, dims, n_per)
    nbrs = []
    for axis in range(3):
        if dims[axis] == 1:
            nbrs.append((None, None))
            continue
        def at(step):
            c = list(coord); c[axis] = (c[axis] + step) % dims[axis]
            return int(np.ravel_multi_index(tuple(c), dims))
        nbrs.append((at(-1), at(+1)))
    lp = OracleLP(state)
    n = X.exchange(lp, lo, hi, nbrs)
    assert n == lp.state[0].shape[0]
    torch.save({"state": lp.state, "lo": lo, "hi": hi}, os.path.join(out, "r%d.pt" % rank))
    dist.barrier()
    dist.destroy_process_group()


def serial_reference(dims, n_per):
    """The same three sweeps done in one process, neighbour buffers handed over directly."""
    from oracle import lp_oracle as orc
    ranks = list(itertools.product(*[range(d) for d in dims]))
    faces = [np.linspace(GLO, GHI, d + 1) for d in dims]
    state = {rk: initial_state(rk, dims, n_per)[0] for rk in ranks}
    for axis in range(3):
        packed = {rk: orc.migrate_pack(axis, faces[axis][rk[axis]], faces[axis][rk[axis] + 1], GLO, GHI, 1, *state[rk])
                  for rk in ranks}
        for rk in ranks:
            def nb(step):
                c = list(rk); c[axis] = (c[axis] + step) % dims[axis]; return tuple(c)
            fl = packed[nb(-1)][3] if dims[axis] > 1 else None
            fr = packed[nb(+1)][2] if dims[axis] > 1 else None
            state[rk] = orc.migrate_unpack(packed[rk][1], fl, fr, *state[rk])
    return state


def _run(dims, n_per, tmp_path):
    world = int(np.prod(dims))
    port = 29500 + (os.getpid() * 7 + world) % 2000
    mp.spawn(_rank_main, args=(dims, n_per, port, str(tmp_path)), nprocs=world, join=True)
    want = serial_reference(dims, n_per)
    seen = []
    for rank in range(world):
        r = torch.load(os.path.join(str(tmp_path), "r%d.pt" % rank), weights_only=False)
        coord = tuple(int(c) for c in np.unravel_index(rank, dims))
        for g, w in zip(r["state"], want[coord]):
            assert np.array_equal(g, w)
        pos = np.stack(r["state"][:3], axis=1)
        assert (pos >= r["lo"]).all() and (pos < r["hi"]).all()          # everybody at home
        seen += r["state"][3].tolist()
    assert sorted(seen) == list(range(world * n_per))


def test_two_ranks_one_periodic_axis(tmp_path):
    _run((2, 1, 1), 400, tmp_path)          # left and right neighbour are the same rank


def test_four_ranks_two_axes(tmp_path):
    _run((2, 1, 2), 300, tmp_path)
