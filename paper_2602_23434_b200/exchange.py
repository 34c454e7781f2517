"""Host plumbing of the particle exchange between ranks: torch.distributed point-to-point
calls around lp_migrate_count / _pack / _unpack.  No arithmetic of the method lives here -- the destination
rule, the packing and the hole filling run in the CUDA kernels (lp_migrate.cu); this module sizes the buffers
from the exchanged counts and moves them (NCCL over NVLink for CUDA tensors; any backend torch.distributed
offers for the tensors `lp.migrate_buffer` returns)."""
import torch
import torch.distributed as dist


def exchange_direction(lp, axis, lo, hi, left, right, group=None):
    """One directional sweep for this rank, which owns [lo, hi) along `axis`.  `left` / `right`: the ranks of
    the two neighbours (None: no neighbour on that side; both may be the same rank on a periodic axis cut in
    two).  Steps 1-8 of PAPER.md:201-214: count, post receives, size buffers, pack, send, grow the particle
    arrays by whole chunks if the arrivals do not fit, wait, unpack.  Returns the new particle count."""
    n_left, n_right = lp.migrate_count(axis, lo, hi)                      # step 1
    if (left is None and n_left) or (right is None and n_right):
        raise RuntimeError("particles leave through a side without a neighbour (delete them first: lp_compact)")
    dev = lp.migrate_buffer(0).device
    send_l = torch.tensor([n_left], dtype=torch.int64, device=dev)
    send_r = torch.tensor([n_right], dtype=torch.int64, device=dev)
    recv_l = torch.zeros(1, dtype=torch.int64, device=dev)               # what the left neighbour sends right
    recv_r = torch.zeros(1, dtype=torch.int64, device=dev)
    _p2p([(send_l, left), (send_r, right)], [(recv_r, right), (recv_l, left)], group)
    n_from_left, n_from_right = int(recv_l.item()), int(recv_r.item())
    in_l, in_r = lp.migrate_buffer(n_from_left), lp.migrate_buffer(n_from_right)      # steps 2-3
    out_l, out_r = lp.migrate_pack(n_left, n_right)                       # step 4
    surplus = n_from_left + n_from_right - (n_left + n_right)
    if surplus > 0 and hasattr(lp, "reserve"):
        lp.reserve(surplus)                                               # step 6 (no-op while the capacity suffices)
    _p2p([(out_l, left if n_left else None), (out_r, right if n_right else None)],
         [(in_r, right if n_from_right else None), (in_l, left if n_from_left else None)], group)    # steps 5, 7
    return lp.migrate_unpack(in_l, n_from_left, in_r, n_from_right)       # steps 6, 8


def _p2p(sends, recvs, group):
    """Leftward messages first, then rightward ones, on both sides: with one peer on both sides (two ranks on a
    periodic axis) the k-th send to it meets its k-th receive from us."""
    ops = [dist.P2POp(dist.isend, t, peer, group) for t, peer in sends if peer is not None]
    ops += [dist.P2POp(dist.irecv, t, peer, group) for t, peer in recvs if peer is not None]
    if ops:
        for req in dist.batch_isend_irecv(ops):
            req.wait()


def exchange(lp, box_lo, box_hi, neighbours, group=None):
    """The three directional sweeps (x, then y, then z).  box_lo / box_hi: this rank's sub-box;
    neighbours[axis] = (left rank or None, right rank or None).  Returns the new particle count."""
    n = None
    for axis in range(3):
        left, right = neighbours[axis]
        n = exchange_direction(lp, axis, box_lo[axis], box_hi[axis], left, right, group)
    return n
