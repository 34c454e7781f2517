"""ctypes binding of include/lp.h -- same names, argument marshalling only.

Every step of the path runs in the CUDA kernels of liblp_b200.so; this module never computes.
It fails loudly (ImportError / LPError) when the library cannot be built or loaded: there is
no CPU fallback.  PyTorch appears only in `LP`, the convenience holder that keeps the device
tensors alive and hands their data_ptr() and the current stream to the C ABI.
"""
import ctypes as C
import os

from . import build as _build

LP_OK, LP_ERR_INVALID_ARG, LP_ERR_STATE, LP_ERR_CUDA, LP_ERR_UNSUPPORTED, LP_ERR_WORKSPACE = 0, -1, -2, -3, -4, -5
_STATUS_NAMES = {0: "LP_OK", -1: "LP_ERR_INVALID_ARG", -2: "LP_ERR_STATE", -3: "LP_ERR_CUDA",
                 -4: "LP_ERR_UNSUPPORTED", -5: "LP_ERR_WORKSPACE"}

EXPORTS = ("lp_create", "lp_destroy", "lp_last_error", "lp_workspace_bytes", "lp_bind_workspace",
           "lp_bind_particles", "lp_bind_diag", "lp_set_fields", "lp_interpolate", "lp_sort", "lp_push",
           "lp_spectral_update", "lp_step", "lp_step_host", "lp_get_diag", "lp_launch_count", "lp_get_bins",
           "lp_timing_enable", "lp_timing_read", "lp_get_cfl_bins", "lp_shock_update", "lp_compact", "lp_push_rk3", "lp_chunked_capacity", "lp_set_count",
           "lp_set_pingpong", "lp_current_particles",
           "lp_migrate_record_bytes", "lp_migrate_count", "lp_migrate_pack", "lp_migrate_unpack",
           "lp_capacity", "lp_workspace_bytes_for", "lp_rebind",
           "lp_bind_energy_grid", "lp_init_energy_grid", "lp_rebind_energy_grid", "lp_current_energy_grid",
           "lp_interpolate_tiled", "lp_number_static", "lp_set_cap_policy")


class LPError(RuntimeError):
    def __init__(self, status, detail=""):
        self.status = status
        super().__init__("%s (%d)%s" % (_STATUS_NAMES.get(status, "?"), status, (": " + detail) if detail else ""))


class lp_config(C.Structure):
    _fields_ = [("struct_size", C.c_uint32),
                ("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32),
                ("xlo", C.c_double * 3), ("xhi", C.c_double * 3), ("periodic", C.c_int32 * 3),
                ("np", C.c_int64), ("nbins", C.c_int32),
                ("e_min", C.c_double), ("e_max", C.c_double),
                ("kappa", C.c_double), ("u_rad", C.c_double), ("cfl_e", C.c_double),
                ("max_substeps", C.c_int32), ("sort_every", C.c_int32), ("device", C.c_int32)]


class lp_diag(C.Structure):
    _fields_ = [("np", C.c_int64), ("sum_substeps", C.c_int64), ("max_substeps", C.c_int32),
                ("n_capped", C.c_int64), ("n_outside", C.c_int64), ("number", C.c_double),
                ("lost", C.c_double), ("steps", C.c_int64), ("sorts", C.c_int64)]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


_lib = None


def library_path():
    return _build.LIB


def load():
    """Build (if stale) and load liblp_b200.so; raises if that is impossible."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.build()
    lib = C.CDLL(path)
    vp, dp = C.c_void_p, C.c_void_p
    lib.lp_create.argtypes = [C.POINTER(lp_config), C.POINTER(vp)]
    lib.lp_destroy.argtypes = [vp]
    lib.lp_last_error.argtypes = [vp]
    lib.lp_last_error.restype = C.c_char_p
    lib.lp_workspace_bytes.argtypes = [C.POINTER(lp_config), C.POINTER(C.c_size_t)]
    lib.lp_bind_workspace.argtypes = [vp, dp, C.c_size_t]
    lib.lp_bind_particles.argtypes = [vp, dp, dp, dp, dp, dp]
    lib.lp_bind_diag.argtypes = [vp, dp, dp]
    lib.lp_set_fields.argtypes = [vp] + [dp] * 7 + [vp]
    lib.lp_interpolate.argtypes = [vp, dp, dp, vp]
    lib.lp_interpolate_tiled.argtypes = [vp, dp, vp]
    lib.lp_sort.argtypes = [vp, vp]
    lib.lp_push.argtypes = [vp, C.c_double, C.c_int, vp]
    lib.lp_spectral_update.argtypes = [vp, C.c_double, vp]
    lib.lp_step.argtypes = [vp, C.c_double, vp]
    lib.lp_shock_update.argtypes = [vp, vp, C.c_double, vp]
    lib.lp_compact.argtypes = [vp, vp, C.POINTER(C.c_int64), vp]
    lib.lp_push_rk3.argtypes = [vp, C.c_double, C.c_int, vp]
    lib.lp_chunked_capacity.argtypes = [C.c_int64, C.c_int32, C.POINTER(C.c_int64)]
    lib.lp_set_count.argtypes = [vp, C.c_int64]
    lib.lp_step_host.argtypes = [vp, C.c_double, dp, dp, dp, dp, dp, vp]
    lib.lp_get_diag.argtypes = [vp, C.POINTER(lp_diag), vp]
    lib.lp_launch_count.argtypes = [vp, C.POINTER(C.c_int64)]
    lib.lp_get_bins.argtypes = [vp, dp, dp]
    lib.lp_timing_enable.argtypes = [vp, C.c_int]
    lib.lp_get_cfl_bins.argtypes = [vp, C.POINTER(C.c_int32), C.POINTER(C.c_int32)]
    lib.lp_timing_read.argtypes = [vp, C.POINTER(C.c_double), C.POINTER(C.c_int32)]
    lib.lp_set_pingpong.argtypes = [vp, C.c_int, vp]
    lib.lp_current_particles.argtypes = [vp] + [C.POINTER(C.c_void_p)] * 5
    lib.lp_bind_energy_grid.argtypes = [vp, dp, dp]
    lib.lp_init_energy_grid.argtypes = [vp, C.c_int64, C.c_int64, vp]
    lib.lp_rebind_energy_grid.argtypes = [vp, dp, dp, vp]
    lib.lp_current_energy_grid.argtypes = [vp, C.POINTER(C.c_void_p)]
    lib.lp_capacity.argtypes = [vp, C.POINTER(C.c_int64)]
    lib.lp_workspace_bytes_for.argtypes = [vp, C.c_int64, C.POINTER(C.c_size_t)]
    lib.lp_rebind.argtypes = [vp, C.c_int64, dp, C.c_size_t, dp, dp, dp, dp, dp, vp]
    lib.lp_migrate_record_bytes.argtypes = [vp, C.POINTER(C.c_size_t)]
    lib.lp_migrate_count.argtypes = [vp, C.c_int, C.c_double, C.c_double, C.POINTER(C.c_int64), C.POINTER(C.c_int64), vp]
    lib.lp_migrate_pack.argtypes = [vp, dp, dp, vp]
    lib.lp_migrate_unpack.argtypes = [vp, dp, C.c_int64, dp, C.c_int64, C.POINTER(C.c_int64), vp]
    lib.lp_set_cap_policy.argtypes = [vp, C.c_int]
    lib.lp_number_static.argtypes = [C.c_int, dp, dp, C.c_int32, C.c_int64, dp, vp, C.c_char_p, C.c_size_t]
    for name in EXPORTS:
        if name != "lp_last_error":
            getattr(lib, name).restype = C.c_int
    _lib = lib
    return lib


def _check(ctx, st):
    if st != LP_OK:
        detail = load().lp_last_error(ctx).decode() if ctx else ""
        raise LPError(st, detail)


def make_config(nx, ny, nz, xlo, xhi, periodic, np, nbins, e_min, e_max, kappa=1.0, u_rad=0.0,
                cfl_e=0.5, max_substeps=4096, sort_every=0, device=0):
    c = lp_config()
    c.struct_size = C.sizeof(lp_config)
    c.nx, c.ny, c.nz = int(nx), int(ny), int(nz)
    for d in range(3):
        c.xlo[d] = float(xlo[d]); c.xhi[d] = float(xhi[d]); c.periodic[d] = int(periodic[d])
    c.np, c.nbins = int(np), int(nbins)
    c.e_min, c.e_max = float(e_min), float(e_max)
    c.kappa, c.u_rad, c.cfl_e = float(kappa), float(u_rad), float(cfl_e)
    c.max_substeps, c.sort_every, c.device = int(max_substeps), int(sort_every), int(device)
    return c


# ---- the C ABI, one Python function per entry point (pointers are ints / None) -------------

def lp_create(cfg):
    out = C.c_void_p()
    st = load().lp_create(C.byref(cfg), C.byref(out))
    if st != LP_OK:
        detail = load().lp_last_error(out).decode() if out else ""
        if out:
            load().lp_destroy(out)
        raise LPError(st, detail)
    return out


def lp_destroy(ctx):
    _check(None, load().lp_destroy(ctx))


def lp_last_error(ctx):
    return load().lp_last_error(ctx).decode()


def lp_workspace_bytes(cfg):
    out = C.c_size_t()
    _check(None, load().lp_workspace_bytes(C.byref(cfg), C.byref(out)))
    return out.value


def lp_bind_workspace(ctx, ptr, nbytes):
    _check(ctx, load().lp_bind_workspace(ctx, ptr, nbytes))


def lp_bind_particles(ctx, x, y, z, pid, chi):
    _check(ctx, load().lp_bind_particles(ctx, x, y, z, pid, chi))


def lp_bind_diag(ctx, nsub, lost):
    _check(ctx, load().lp_bind_diag(ctx, nsub, lost))


def lp_set_fields(ctx, vx, vy, vz, bx, by, bz, rho, stream=None):
    _check(ctx, load().lp_set_fields(ctx, vx, vy, vz, bx, by, bz, rho, stream))


def lp_interpolate(ctx, out7, cell_key, stream=None):
    _check(ctx, load().lp_interpolate(ctx, out7, cell_key, stream))


def lp_interpolate_tiled(ctx, out7, stream=None):
    _check(ctx, load().lp_interpolate_tiled(ctx, out7, stream))


def lp_sort(ctx, stream=None):
    _check(ctx, load().lp_sort(ctx, stream))


def lp_push(ctx, dt, stage, stream=None):
    _check(ctx, load().lp_push(ctx, float(dt), int(stage), stream))


def lp_spectral_update(ctx, dt, stream=None):
    _check(ctx, load().lp_spectral_update(ctx, float(dt), stream))


def lp_shock_update(ctx, r_ptr, q_r, stream=None):
    _check(ctx, load().lp_shock_update(ctx, r_ptr, float(q_r), stream))


def lp_chunked_capacity(n, e=18):
    cap = C.c_int64()
    st = load().lp_chunked_capacity(int(n), int(e), C.byref(cap))
    if st != LP_OK:
        raise LPError(st)
    return int(cap.value)


def lp_set_count(ctx, n):
    _check(ctx, load().lp_set_count(ctx, int(n)))


def lp_push_rk3(ctx, dt, stage, stream=None):
    _check(ctx, load().lp_push_rk3(ctx, float(dt), int(stage), stream))


def lp_compact(ctx, flag_ptr, stream=None):
    n = C.c_int64()
    _check(ctx, load().lp_compact(ctx, flag_ptr, C.byref(n), stream))
    return int(n.value)


def lp_migrate_record_bytes(ctx):
    out = C.c_size_t()
    _check(ctx, load().lp_migrate_record_bytes(ctx, C.byref(out)))
    return out.value


def lp_migrate_count(ctx, axis, lo, hi, stream=None):
    nl = C.c_int64(); nr = C.c_int64()
    _check(ctx, load().lp_migrate_count(ctx, int(axis), float(lo), float(hi), C.byref(nl), C.byref(nr), stream))
    return int(nl.value), int(nr.value)


def lp_migrate_pack(ctx, buf_left, buf_right, stream=None):
    _check(ctx, load().lp_migrate_pack(ctx, buf_left, buf_right, stream))


def lp_migrate_unpack(ctx, from_left, n_from_left, from_right, n_from_right, stream=None):
    n = C.c_int64()
    _check(ctx, load().lp_migrate_unpack(ctx, from_left, int(n_from_left), from_right, int(n_from_right), C.byref(n), stream))
    return int(n.value)


def lp_bind_energy_grid(ctx, eng, eng_scratch=None):
    _check(ctx, load().lp_bind_energy_grid(ctx, eng, eng_scratch))


def lp_init_energy_grid(ctx, first, count, stream=None):
    _check(ctx, load().lp_init_energy_grid(ctx, int(first), int(count), stream))


def lp_rebind_energy_grid(ctx, eng, eng_scratch=None, stream=None):
    _check(ctx, load().lp_rebind_energy_grid(ctx, eng, eng_scratch, stream))


def lp_current_energy_grid(ctx):
    p = C.c_void_p()
    _check(ctx, load().lp_current_energy_grid(ctx, C.byref(p)))
    return p.value or 0


def lp_capacity(ctx):
    out = C.c_int64()
    _check(ctx, load().lp_capacity(ctx, C.byref(out)))
    return int(out.value)


def lp_workspace_bytes_for(ctx, capacity):
    out = C.c_size_t()
    _check(ctx, load().lp_workspace_bytes_for(ctx, int(capacity), C.byref(out)))
    return out.value


def lp_rebind(ctx, capacity, workspace, nbytes, x, y, z, pid, chi, stream=None):
    _check(ctx, load().lp_rebind(ctx, int(capacity), workspace, nbytes, x, y, z, pid, chi, stream))


def lp_set_pingpong(ctx, enable, stream=None):
    _check(ctx, load().lp_set_pingpong(ctx, int(bool(enable)), stream))


def lp_current_particles(ctx):
    """Device addresses (ints) of x, y, z, id, chi as they are now."""
    p = [C.c_void_p() for _ in range(5)]
    _check(ctx, load().lp_current_particles(ctx, *[C.byref(q) for q in p]))
    return tuple(q.value or 0 for q in p)


def lp_step(ctx, dt, stream=None):
    _check(ctx, load().lp_step(ctx, float(dt), stream))


def lp_step_host(ctx, dt, hx, hy, hz, hid, hchi, stream=None):
    _check(ctx, load().lp_step_host(ctx, float(dt), hx, hy, hz, hid, hchi, stream))


def lp_get_diag(ctx, stream=None):
    d = lp_diag()
    _check(ctx, load().lp_get_diag(ctx, C.byref(d), stream))
    return d.as_dict()


def lp_set_cap_policy(ctx, error_on_cap):
    _check(ctx, load().lp_set_cap_policy(ctx, int(bool(error_on_cap))))


def lp_launch_count(ctx):
    out = C.c_int64()
    _check(ctx, load().lp_launch_count(ctx, C.byref(out)))
    return out.value


def lp_get_cfl_bins(ctx):
    bins = (C.c_int32 * 64)(); n = C.c_int32()
    _check(ctx, load().lp_get_cfl_bins(ctx, bins, C.byref(n)))
    return None if n.value < 0 else [bins[k] for k in range(n.value)]


def lp_timing_enable(ctx, max_records):
    _check(ctx, load().lp_timing_enable(ctx, int(max_records)))


def lp_timing_read(ctx):
    ms = C.c_double(); n = C.c_int32()
    _check(ctx, load().lp_timing_read(ctx, C.byref(ms), C.byref(n)))
    return ms.value, n.value


def lp_number_static(device, chi_ptr, widths_ptr, nbins, np_, number_ptr, stream=None):
    """The allocation-free particle number (include/lp.h): device pointers in, one double written at number_ptr on
    `stream`.  Needs no context; the reason of a refusal comes back in the exception."""
    err = C.create_string_buffer(256)
    st = load().lp_number_static(int(device), chi_ptr, widths_ptr, int(nbins), int(np_), number_ptr, stream, err, len(err))
    if st != LP_OK:
        raise LPError(st, err.value.decode())


def lp_get_bins(ctx, nbins):
    import numpy as np
    E = np.empty(nbins + 1); dE = np.empty(nbins)
    _check(ctx, load().lp_get_bins(ctx, E.ctypes.data, dE.ctypes.data))
    return E, dE
