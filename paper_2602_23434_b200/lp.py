"""`LP`: a thin holder around one lp_ctx that owns the torch device tensors (memory and stream
plumbing only) and forwards to the C ABI.  No arithmetic of the method lives here."""
import torch

from . import binding as B


class LP:
    def __init__(self, cfg, device=None):
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2602_23434_b200 needs a CUDA device (sm_100a); there is no CPU path")
        self.cfg = cfg
        self.device = torch.device("cuda", cfg.device) if device is None else torch.device(device)
        B.load()
        self.ctx = B.lp_create(cfg)
        nbytes = B.lp_workspace_bytes(cfg)
        self.workspace, ptr = self._alloc_workspace(nbytes)
        B.lp_bind_workspace(self.ctx, ptr, nbytes)
        self.workspace_bytes = nbytes
        self._bound = None            # the caller-side tensors x, y, z, id, chi (the bound arrays)
        self.capacity = cfg.np
        self.nsub = self.lost = None
        self._eng = self._eng_scratch = None
        self._fields = None

    def _alloc_workspace(self, nbytes):
        ws = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
        return ws, ws.data_ptr() + (-ws.data_ptr()) % 256

    def close(self):
        if self.ctx is not None:
            torch.cuda.synchronize(self.device)
            B.lp_destroy(self.ctx)
            self.ctx = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    @property
    def stream(self):
        return torch.cuda.current_stream(self.device).cuda_stream

    def _dev(self, a, dtype):
        t = torch.as_tensor(a)
        if dtype == torch.uint64 and t.dtype != torch.uint64:
            t = t.to(torch.int64).view(torch.uint64) if t.dtype == torch.int64 else t
        return t.to(device=self.device, dtype=dtype).contiguous()

    def bind_particles(self, x, y, z, pid, chi):
        import numpy as np
        n, nb = self.cfg.np, self.cfg.nbins
        bx = self._dev(x, torch.float64); by = self._dev(y, torch.float64); bz = self._dev(z, torch.float64)
        pid = torch.as_tensor(np.ascontiguousarray(pid).view(np.int64)) if not torch.is_tensor(pid) else pid
        bid = pid.to(self.device).contiguous()
        bchi = self._dev(chi, torch.float64)
        assert bx.numel() == n and bchi.shape == (n, nb) and bid.numel() == n
        B.lp_bind_particles(self.ctx, bx.data_ptr(), by.data_ptr(), bz.data_ptr(), bid.data_ptr(), bchi.data_ptr())
        self._bound = (bx, by, bz, bid, bchi)

    def set_pingpong(self, enable=True):
        """Let a re-sort leave the state in the workspace twins of the bound arrays (no copy back): x, y, z,
        id, chi of this object then follow lp_current_particles."""
        B.lp_set_pingpong(self.ctx, enable, self.stream)

    def _view(self, ptr, elems, dtype):
        """A tensor over `elems` elements of the workspace starting at device address ptr (no copy)."""
        off = ptr - self.workspace.data_ptr()
        assert 0 <= off and off + elems * 8 <= self.workspace.numel()
        return self.workspace[off: off + elems * 8].view(dtype)

    def current(self):
        """The tensors that hold the particle state now: (x, y, z, id, chi) -- the bound ones, or (ping-pong,
        after a re-sort) views of their workspace twins.  Length = the capacity the context was created with."""
        ptrs = B.lp_current_particles(self.ctx)
        if ptrs[0] == self._bound[0].data_ptr():
            return self._bound
        n, nb = self.capacity, self.cfg.nbins
        return (self._view(ptrs[0], n, torch.float64), self._view(ptrs[1], n, torch.float64),
                self._view(ptrs[2], n, torch.float64), self._view(ptrs[3], n, torch.int64),
                self._view(ptrs[4], n * nb, torch.float64).view(n, nb))

    x = property(lambda self: self.current()[0])
    y = property(lambda self: self.current()[1])
    z = property(lambda self: self.current()[2])
    id = property(lambda self: self.current()[3])
    chi = property(lambda self: self.current()[4])

    def bind_diag(self, nsub=True, lost=True):
        n = self.capacity
        self.nsub = torch.zeros(n, dtype=torch.int32, device=self.device) if nsub else None
        self.lost = torch.zeros(n, dtype=torch.float64, device=self.device) if lost else None
        B.lp_bind_diag(self.ctx, self.nsub.data_ptr() if nsub else None, self.lost.data_ptr() if lost else None)

    def set_fields(self, fields7):
        f = [self._dev(t, torch.float64) for t in fields7]
        ncell = self.cfg.nx * self.cfg.ny * self.cfg.nz
        assert len(f) == 7 and all(t.numel() == ncell for t in f)
        B.lp_set_fields(self.ctx, *[t.data_ptr() for t in f], self.stream)
        self._fields = f          # keep alive until the stream has consumed them

    def interpolate(self, want_fields=True, want_key=True):
        n = self.cfg.np
        out7 = torch.empty((7, n), dtype=torch.float64, device=self.device) if want_fields else None
        key = torch.empty(n, dtype=torch.int32, device=self.device) if want_key else None
        B.lp_interpolate(self.ctx, out7.data_ptr() if want_fields else None,
                         key.data_ptr() if want_key else None, self.stream)
        return out7, key

    def interpolate_tiled(self):
        """lp_interpolate's fields through shared-memory tiles (for sets sorted by cell); same values."""
        out7 = torch.empty((7, self.cfg.np), dtype=torch.float64, device=self.device)
        B.lp_interpolate_tiled(self.ctx, out7.data_ptr(), self.stream)
        return out7

    def sort(self):
        B.lp_sort(self.ctx, self.stream)

    def push(self, dt, stage):
        B.lp_push(self.ctx, dt, stage, self.stream)

    def push_rk3(self, dt, stage):
        B.lp_push_rk3(self.ctx, dt, stage, self.stream)

    def spectral_update(self, dt):
        B.lp_spectral_update(self.ctx, dt, self.stream)

    def shock_update(self, r, q_r=0.0):
        """Eq. 7-8 on the rows with r[p] > 1; r: float64 CUDA tensor [np] of compression ratios."""
        assert r.is_cuda and r.dtype == torch.float64 and r.numel() >= self.cfg.np and r.is_contiguous()
        B.lp_shock_update(self.ctx, r.data_ptr(), q_r, self.stream)

    def set_count(self, n):
        """Use the first n particles of the bound arrays (n <= the capacity the context was created with)."""
        B.lp_set_count(self.ctx, n)
        self.cfg.np = n            # (the binding's copy of the count sizes the outputs of interpolate)

    # ---- per-particle moving energy grid (Listing 3's eng_; readings E1-E4 of DESIGN.md)
    def bind_energy_grid(self, init=True, sortable=True):
        """Switch to the moving energy grid: allocates eng [capacity][nbins+1] (and the scratch a sort needs),
        starts every particle on the fixed table's edges."""
        shape = (self.capacity, self.cfg.nbins + 1)
        self._eng = torch.empty(shape, dtype=torch.float64, device=self.device)
        self._eng_scratch = torch.empty(shape, dtype=torch.float64, device=self.device) if sortable else None
        B.lp_bind_energy_grid(self.ctx, self._eng.data_ptr(), self._eng_scratch.data_ptr() if sortable else None)
        if init:
            B.lp_init_energy_grid(self.ctx, 0, self.capacity, self.stream)
        return self._eng

    @property
    def eng(self):
        """The tensor that holds the energy grid now (with ping-pong buffers a re-sort swaps it with the scratch)."""
        if self._eng is None:
            return None
        ptr = B.lp_current_energy_grid(self.ctx)
        return self._eng if ptr == self._eng.data_ptr() else self._eng_scratch

    def unbind_energy_grid(self):
        B.lp_bind_energy_grid(self.ctx, None, None)
        self._eng = self._eng_scratch = None

    # ---- chunked growth (Listing 1; Reserve() / Shrink() of Listing 2)
    def _rebind(self, capacity):
        n, nb = self.cfg.np, self.cfg.nbins
        f64 = lambda *shape: torch.empty(shape, dtype=torch.float64, device=self.device)
        new = (f64(capacity), f64(capacity), f64(capacity),
               torch.empty(capacity, dtype=torch.int64, device=self.device), f64(capacity, nb))
        nbytes = B.lp_workspace_bytes_for(self.ctx, capacity)
        ws, ptr = self._alloc_workspace(nbytes)
        B.lp_rebind(self.ctx, capacity, ptr, nbytes, *[t.data_ptr() for t in new], self.stream)
        # the old tensors stay referenced until the stream has passed the copies
        self._retired = (self._bound, self.workspace, self.nsub, self.lost)
        self._bound, self.workspace, self.workspace_bytes, self.capacity = new, ws, nbytes, capacity
        had = (self.nsub is not None, self.lost is not None)
        self.nsub = self.lost = None
        if any(had):
            self.bind_diag(*had)
        if self._eng is not None:                            # the energy grid follows: new arrays, rows copied over
            shape = (capacity, nb + 1)
            eng = torch.empty(shape, dtype=torch.float64, device=self.device)
            scr = torch.empty(shape, dtype=torch.float64, device=self.device) if self._eng_scratch is not None else None
            B.lp_rebind_energy_grid(self.ctx, eng.data_ptr(), scr.data_ptr() if scr is not None else None, self.stream)
            self._retired = self._retired + (self._eng, self._eng_scratch)
            self._eng, self._eng_scratch = eng, scr

    def reserve(self, n_new, e=18):
        """Room for n_new more particles behind the current ones (Listing 2's Reserve): when the capacity does
        not suffice, storage for lp_chunked_capacity(count + n_new, e) particles -- whole chunks of 2^e -- is
        allocated and the state moved there (lp_rebind).  Write the new particles into x, y, z, id, chi
        [count : count + n_new] and call set_count.  Returns the capacity."""
        need = self.cfg.np + int(n_new)
        if need > self.capacity:
            self._rebind(B.lp_chunked_capacity(need, e))
        return self.capacity

    def shrink(self, e=18):
        """Release the trailing chunks that hold no particle (Listing 2's Shrink).  Returns the capacity."""
        cap = max(B.lp_chunked_capacity(self.cfg.np, e), 1 << e)
        if cap < self.capacity:
            self._rebind(cap)
        return self.capacity

    def compact(self, flag=None):
        """Delete the flagged particles (int32 CUDA tensor [np], nonzero = delete; None = those outside the
        box after the last push) and fill the holes from the tail; returns the new particle count.  The
        tensors keep their size: the first `count` entries are the particles."""
        if flag is not None:
            assert flag.is_cuda and flag.dtype == torch.int32 and flag.is_contiguous()
        n = B.lp_compact(self.ctx, flag.data_ptr() if flag is not None else None, self.stream)
        self.cfg.np = n
        return n

    # ---- particle exchange across rank interfaces: count -> pack -> (move buffers) -> unpack
    def migrate_count(self, axis, lo, hi):
        """(n_left, n_right): particles leaving [lo, hi) along `axis` towards the left / right neighbour."""
        return B.lp_migrate_count(self.ctx, axis, lo, hi, self.stream)

    def migrate_buffer(self, n):
        """An (uninitialised) send / receive buffer for n particles: uint8 CUDA tensor, n * (32 + 8 nbins) bytes."""
        return torch.empty(max(1, n) * B.lp_migrate_record_bytes(self.ctx), dtype=torch.uint8, device=self.device)

    def migrate_pack(self, n_left, n_right):
        """Packs the leavers counted by migrate_count; returns (buf_left, buf_right)."""
        bl, br = self.migrate_buffer(n_left), self.migrate_buffer(n_right)
        B.lp_migrate_pack(self.ctx, bl.data_ptr() if n_left else None, br.data_ptr() if n_right else None, self.stream)
        return bl, br

    def migrate_unpack(self, from_left, n_from_left, from_right, n_from_right):
        """Arrivals into the holes / behind the last particle; returns the new particle count."""
        n = B.lp_migrate_unpack(self.ctx, from_left.data_ptr() if n_from_left else None, n_from_left,
                                from_right.data_ptr() if n_from_right else None, n_from_right, self.stream)
        self._keep = (from_left, from_right)      # alive until the stream has consumed them
        self.cfg.np = n
        return n

    def step(self, dt):
        B.lp_step(self.ctx, dt, self.stream)

    def step_host(self, dt, hx, hy, hz, hid, hchi):
        B.lp_step_host(self.ctx, dt, hx.data_ptr(), hy.data_ptr(), hz.data_ptr(), hid.data_ptr(),
                       hchi.data_ptr(), self.stream)

    def diag(self):
        return B.lp_get_diag(self.ctx, self.stream)

    def launch_count(self):
        return B.lp_launch_count(self.ctx)

    def bins(self):
        return B.lp_get_bins(self.ctx, self.cfg.nbins)


def config_from_workload(w, u_rad=0.0, device=0, np=None):
    """lp_config for an lp_inputs.LPWorkload (duck-typed: only attributes are read)."""
    return B.make_config(w.n, w.n, w.n, w.xlo, w.xhi, w.periodic, w.np if np is None else np, w.nbins,
                         w.e_min, w.e_max, kappa=w.kappa, u_rad=u_rad, cfl_e=w.cfl_e,
                         max_substeps=w.max_substeps, sort_every=w.sort_every, device=device)
