"""ctypes wrapper around oracle/lp_oracle.c (numpy in, numpy out).

TEST INFRASTRUCTURE: see oracle/__init__.py.  Argument marshalling only; every
number is computed by the C file.  Names follow lp_oracle.c.
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

FIELD_ORDER = ("vx", "vy", "vz", "bx", "by", "bz", "rho")


class OrcParams(C.Structure):
    _fields_ = [
        ("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32),
        ("xlo", C.c_double * 3), ("xhi", C.c_double * 3),
        ("periodic", C.c_int32 * 3),
        ("nbins", C.c_int32),
        ("e_min", C.c_double), ("e_max", C.c_double),
        ("kappa", C.c_double), ("u_rad", C.c_double),
        ("cfl_e", C.c_double),
        ("max_substeps", C.c_int32),
    ]


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        _lib.orc_row_number.restype = C.c_double
        _lib.orc_cfl_nsub.restype = C.c_int32
    return _lib


def make_params(nx, ny, nz, xlo, xhi, periodic, nbins, e_min, e_max,
                kappa=1.0, u_rad=0.0, cfl_e=0.5, max_substeps=4096):
    p = OrcParams()
    p.nx, p.ny, p.nz = int(nx), int(ny), int(nz)
    for d in range(3):
        p.xlo[d] = float(xlo[d]); p.xhi[d] = float(xhi[d]); p.periodic[d] = int(periodic[d])
    p.nbins = int(nbins)
    p.e_min, p.e_max = float(e_min), float(e_max)
    p.kappa, p.u_rad, p.cfl_e = float(kappa), float(u_rad), float(cfl_e)
    p.max_substeps = int(max_substeps)
    return p


def _d(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a, a.ctypes.data_as(C.POINTER(C.c_double))


def _fields(fields7):
    """fields7: sequence of 7 arrays [nz,ny,nx] in FIELD_ORDER -> (keepalive, double**)."""
    keep = [np.ascontiguousarray(f, dtype=np.float64) for f in fields7]
    assert len(keep) == 7
    arr = (C.POINTER(C.c_double) * 7)(*[k.ctypes.data_as(C.POINTER(C.c_double)) for k in keep])
    return keep, arr


def bin_table(nbins, e_min, e_max):
    E = np.empty(nbins + 1); dE = np.empty(nbins); Ec = np.empty(nbins)
    lib().orc_bin_table(C.c_int32(nbins), C.c_double(e_min), C.c_double(e_max),
                        E.ctypes.data_as(C.POINTER(C.c_double)),
                        dE.ctypes.data_as(C.POINTER(C.c_double)),
                        Ec.ctypes.data_as(C.POINTER(C.c_double)))
    return E, dE, Ec


def cell_key(prm, x, y, z):
    x, px = _d(x); y, py = _d(y); z, pz = _d(z)
    key = np.empty(x.shape[0], dtype=np.uint32)
    lib().orc_cell_key(C.byref(prm), C.c_int64(x.shape[0]), px, py, pz,
                       key.ctypes.data_as(C.POINTER(C.c_uint32)))
    return key


def sort_perm(key, pid):
    key = np.ascontiguousarray(key, dtype=np.uint32)
    pid = np.ascontiguousarray(pid, dtype=np.uint64)
    perm = np.empty(key.shape[0], dtype=np.int64)
    lib().orc_sort_perm(C.c_int64(key.shape[0]), key.ctypes.data_as(C.POINTER(C.c_uint32)),
                        pid.ctypes.data_as(C.POINTER(C.c_uint64)),
                        perm.ctypes.data_as(C.POINTER(C.c_int64)))
    return perm


def gather(prm, fields7, x, y, z):
    keep, fa = _fields(fields7)
    x, px = _d(x); y, py = _d(y); z, pz = _d(z)
    out = np.empty((7, x.shape[0]))
    lib().orc_gather(C.byref(prm), fa, C.c_int64(x.shape[0]), px, py, pz,
                     out.ctypes.data_as(C.POINTER(C.c_double)))
    return out


def push_stage0(prm, fields7, x, y, z, dt, nthreads=1):
    keep, fa = _fields(fields7)
    x, px = _d(x); y, py = _d(y); z, pz = _d(z)
    n = x.shape[0]
    k1 = np.empty((3, n)); rho_old = np.empty(n); xs = np.empty((3, n))
    lib().orc_push_stage0(C.byref(prm), fa, C.c_int64(n), px, py, pz, C.c_double(dt),
                          k1.ctypes.data_as(C.POINTER(C.c_double)),
                          rho_old.ctypes.data_as(C.POINTER(C.c_double)),
                          xs.ctypes.data_as(C.POINTER(C.c_double)), C.c_int32(nthreads))
    return k1, rho_old, xs


def push_stage1(prm, fields7, x, y, z, xs, k1, dt, nthreads=1):
    """Returns new (x, y, z, status); inputs are not modified."""
    keep, fa = _fields(fields7)
    x = np.array(x, dtype=np.float64); y = np.array(y, dtype=np.float64); z = np.array(z, dtype=np.float64)
    xs, pxs = _d(xs); k1, pk1 = _d(k1)
    n = x.shape[0]
    status = np.zeros(n, dtype=np.int32)
    dp = lambda a: a.ctypes.data_as(C.POINTER(C.c_double))
    lib().orc_push_stage1(C.byref(prm), fa, C.c_int64(n), dp(x), dp(y), dp(z), pxs, pk1,
                          C.c_double(dt), status.ctypes.data_as(C.POINTER(C.c_int32)),
                          C.c_int32(nthreads))
    return x, y, z, status


def push_rk3(prm, fields_by_stage, x, y, z, dt):
    """One third-order step; fields_by_stage: the seven fields to use at stages 0, 1, 2 (or one set for all).
    Returns (x, y, z, rho_old, status, stage positions [(x1,y1,z1), (x2,y2,z2)])."""
    if not isinstance(fields_by_stage[0], (list, tuple)):
        fields_by_stage = [fields_by_stage] * 3
    x = np.array(x, dtype=np.float64); y = np.array(y, dtype=np.float64); z = np.array(z, dtype=np.float64)
    n = x.shape[0]
    x0 = np.empty((3, n)); rho_old = np.empty(n); status = np.zeros(n, dtype=np.int32)
    dp = lambda a: a.ctypes.data_as(C.POINTER(C.c_double))
    f = lib().orc_push_rk3_stage
    f.restype = None
    mids = []
    for stage in range(3):
        keep, fa = _fields(fields_by_stage[stage])
        f(C.byref(prm), fa, C.c_int64(n), C.c_int32(stage), dp(x), dp(y), dp(z), dp(x0), C.c_double(dt),
          dp(rho_old), status.ctypes.data_as(C.POINTER(C.c_int32)))
        if stage < 2:
            mids.append((x.copy(), y.copy(), z.copy()))
    return x, y, z, rho_old, status, mids


def coefficients(prm, dt, v, B, rho_new, rho_old):
    a = C.c_double(); cr = C.c_double(); dtau = C.c_double()
    v3 = (C.c_double * 3)(*[float(t) for t in v]); b3 = (C.c_double * 3)(*[float(t) for t in B])
    lib().orc_coefficients(C.byref(prm), C.c_double(dt), v3, b3, C.c_double(rho_new),
                           C.c_double(rho_old), C.byref(a), C.byref(cr), C.byref(dtau))
    return a.value, cr.value, dtau.value


def cfl_nsub(E, dE, a, cr, dtau, cfl_e=0.5, max_substeps=4096):
    E, pE = _d(E); dE, pdE = _d(dE)
    lam = C.c_double()
    n = lib().orc_cfl_nsub(C.c_int32(dE.shape[0]), pE, pdE, C.c_double(a), C.c_double(cr),
                           C.c_double(dtau), C.c_double(cfl_e), C.c_int32(max_substeps),
                           C.byref(lam))
    return int(n), lam.value


def spectral_row(E, dE, a, cr, dtau, nsub, chi):
    """Returns (new chi row, lost)."""
    E, pE = _d(E); dE, pdE = _d(dE)
    chi = np.array(chi, dtype=np.float64)
    lost = C.c_double()
    lib().orc_spectral_row(C.c_int32(dE.shape[0]), pE, pdE, C.c_double(a), C.c_double(cr),
                           C.c_double(dtau), C.c_int32(nsub),
                           chi.ctypes.data_as(C.POINTER(C.c_double)), C.byref(lost))
    return chi, lost.value


def shock_row(E, dE, r, q_r, chi):
    """Eq. 7-8 on one row; returns (new row, changed)."""
    E, pE = _d(E); dE, pdE = _d(dE)
    chi = np.array(chi, dtype=np.float64)
    f = lib().orc_shock_row
    f.restype = C.c_int32
    ch = f(C.c_int32(dE.shape[0]), pE, pdE, C.c_double(r), C.c_double(q_r),
           chi.ctypes.data_as(C.POINTER(C.c_double)))
    return chi, bool(ch)


def shock_update(E, dE, r, q_r, chi):
    """Eq. 7-8 on every row of chi [np][nbins] with compression ratios r [np]; returns the new array."""
    E, pE = _d(E); dE, pdE = _d(dE); r, pr = _d(r)
    chi = np.array(chi, dtype=np.float64, order="C")
    f = lib().orc_shock_update
    f.restype = None
    f(C.c_int32(dE.shape[0]), pE, pdE, C.c_int64(chi.shape[0]), pr, C.c_double(q_r),
      chi.ctypes.data_as(C.POINTER(C.c_double)))
    return chi


def shock_update_grid(eng, r, q_r, chi):
    """Eq. 7-8 on every row, each on its own edges eng [np][nbins+1]; returns the new chi."""
    eng = np.ascontiguousarray(eng, dtype=np.float64); r, pr = _d(r)
    chi = np.array(chi, dtype=np.float64, order="C")
    f = lib().orc_shock_update_grid
    f.restype = None
    dp = C.POINTER(C.c_double)
    f(C.c_int32(chi.shape[1]), C.c_int64(chi.shape[0]), eng.ctypes.data_as(dp), pr, C.c_double(q_r), chi.ctypes.data_as(dp))
    return chi


def compact(flag, x, y, z, pid, chi):
    """The paper's delete-and-fill compaction; returns (x, y, z, id, chi) cut to the new count."""
    flag = np.ascontiguousarray(flag, dtype=np.int32)
    x = np.array(x, dtype=np.float64); y = np.array(y, dtype=np.float64); z = np.array(z, dtype=np.float64)
    pid = np.array(pid, dtype=np.uint64)
    chi = np.array(chi, dtype=np.float64, order="C")
    f = lib().orc_compact
    f.restype = C.c_int64
    dp = C.POINTER(C.c_double)
    keep = f(C.c_int64(x.shape[0]), flag.ctypes.data_as(C.POINTER(C.c_int32)), C.c_int32(chi.shape[1]),
             x.ctypes.data_as(dp), y.ctypes.data_as(dp), z.ctypes.data_as(dp),
             pid.ctypes.data_as(C.POINTER(C.c_uint64)), chi.ctypes.data_as(dp))
    return x[:keep], y[:keep], z[:keep], pid[:keep], chi[:keep]


def migrate_dest(x, lo, hi, glo, ghi, periodic):
    f = lib().orc_migrate_dest
    f.restype = C.c_int32
    return int(f(C.c_double(x), C.c_double(lo), C.c_double(hi), C.c_double(glo), C.c_double(ghi), C.c_int32(periodic)))


def migrate_pack(axis, lo, hi, glo, ghi, periodic, x, y, z, pid, chi):
    """Steps 1 and 4 of the exchange along `axis` for the rank owning [lo, hi).  Returns
    (dest [np] int32, holes [n_left+n_right] int64, left buffer, right buffer); a buffer is the tuple
    (x, y, z, id, chi) of the particles sent that way, in ascending index order."""
    x, px = _d(x); y, py = _d(y); z, pz = _d(z)
    pid = np.ascontiguousarray(pid, dtype=np.uint64)
    chi = np.ascontiguousarray(chi, dtype=np.float64)
    n = x.shape[0]
    nb = chi.shape[1]
    dest = np.zeros(n, dtype=np.int32); holes = np.zeros(max(n, 1), dtype=np.int64)
    nl = C.c_int64(); nr = C.c_int64()
    bufs = [[np.zeros(max(n, 1)), np.zeros(max(n, 1)), np.zeros(max(n, 1)), np.zeros(max(n, 1), dtype=np.uint64),
             np.zeros((max(n, 1), nb))] for _ in range(2)]
    dp = C.POINTER(C.c_double); up = C.POINTER(C.c_uint64)
    args = []
    for b in bufs:
        args += [b[0].ctypes.data_as(dp), b[1].ctypes.data_as(dp), b[2].ctypes.data_as(dp), b[3].ctypes.data_as(up),
                 b[4].ctypes.data_as(dp)]
    f = lib().orc_migrate_pack
    f.restype = None
    f(C.c_int64(n), C.c_int32(nb), C.c_int32(axis), C.c_double(lo), C.c_double(hi), C.c_double(glo), C.c_double(ghi),
      C.c_int32(periodic), px, py, pz, pid.ctypes.data_as(up), chi.ctypes.data_as(dp),
      dest.ctypes.data_as(C.POINTER(C.c_int32)), holes.ctypes.data_as(C.POINTER(C.c_int64)),
      C.byref(nl), C.byref(nr), *args)
    left = tuple(a[:nl.value].copy() for a in bufs[0])
    right = tuple(a[:nr.value].copy() for a in bufs[1])
    return dest, holes[:nl.value + nr.value].copy(), left, right


def migrate_unpack(holes, from_left, from_right, x, y, z, pid, chi):
    """Step 8: the arrivals (buffers as returned by migrate_pack of the neighbours; None = nothing) into the
    holes / behind the last particle, the remaining holes compacted away.  Returns (x, y, z, id, chi) of the
    new particle set."""
    nb = np.asarray(chi).shape[1]
    empty = (np.zeros(0), np.zeros(0), np.zeros(0), np.zeros(0, dtype=np.uint64), np.zeros((0, nb)))
    L = from_left if from_left is not None else empty
    R = from_right if from_right is not None else empty
    n = np.asarray(x).shape[0]
    nin = L[0].shape[0] + R[0].shape[0]
    cap = n + nin
    def grow(a, dtype, cols=None):
        out = np.zeros((cap,) if cols is None else (cap, cols), dtype=dtype)
        out[:n] = a
        return out
    x = grow(x, np.float64); y = grow(y, np.float64); z = grow(z, np.float64)
    pid = grow(pid, np.uint64); chi = grow(chi, np.float64, nb)
    holes = np.ascontiguousarray(holes, dtype=np.int64)
    dp = C.POINTER(C.c_double); up = C.POINTER(C.c_uint64)
    def buf(b):
        b = (np.ascontiguousarray(b[0], dtype=np.float64), np.ascontiguousarray(b[1], dtype=np.float64),
             np.ascontiguousarray(b[2], dtype=np.float64), np.ascontiguousarray(b[3], dtype=np.uint64),
             np.ascontiguousarray(b[4], dtype=np.float64))
        return b, [b[0].ctypes.data_as(dp), b[1].ctypes.data_as(dp), b[2].ctypes.data_as(dp), b[3].ctypes.data_as(up),
                   b[4].ctypes.data_as(dp)]
    Lk, La = buf(L); Rk, Ra = buf(R)
    f = lib().orc_migrate_unpack
    f.restype = C.c_int64
    cnt = f(C.c_int64(n), C.c_int32(nb), holes.ctypes.data_as(C.POINTER(C.c_int64)), C.c_int64(holes.shape[0]),
            C.c_int64(Lk[0].shape[0]), *La, C.c_int64(Rk[0].shape[0]), *Ra,
            x.ctypes.data_as(dp), y.ctypes.data_as(dp), z.ctypes.data_as(dp), pid.ctypes.data_as(up),
            chi.ctypes.data_as(dp))
    return x[:cnt], y[:cnt], z[:cnt], pid[:cnt], chi[:cnt]


def moving_row(a, cr, dtau, eng, chi):
    """One step of the moving energy grid on one particle; returns (new edges, new chi)."""
    eng = np.array(eng, dtype=np.float64); chi = np.array(chi, dtype=np.float64)
    f = lib().orc_moving_row
    f.restype = None
    dp = C.POINTER(C.c_double)
    f(C.c_int32(chi.shape[0]), C.c_double(a), C.c_double(cr), C.c_double(dtau), eng.ctypes.data_as(dp),
      chi.ctypes.data_as(dp))
    return eng, chi


def moving_update(prm, fields7, x, y, z, rho_old, dt, eng, chi, nthreads=1):
    """Returns (new eng [np,nbins+1], new chi [np,nbins])."""
    keep, fa = _fields(fields7)
    x, px = _d(x); y, py = _d(y); z, pz = _d(z); rho_old, pr = _d(rho_old)
    eng = np.array(eng, dtype=np.float64, order="C"); chi = np.array(chi, dtype=np.float64, order="C")
    n = x.shape[0]
    assert chi.shape == (n, prm.nbins) and eng.shape == (n, prm.nbins + 1)
    f = lib().orc_moving_update
    f.restype = None
    dp = C.POINTER(C.c_double)
    f(C.byref(prm), fa, C.c_int64(n), px, py, pz, pr, C.c_double(dt), eng.ctypes.data_as(dp), chi.ctypes.data_as(dp),
      C.c_int32(nthreads))
    return eng, chi


def row_number(dE, chi):
    dE, pdE = _d(dE); chi, pchi = _d(chi)
    return float(lib().orc_row_number(C.c_int32(dE.shape[0]), pdE, pchi))


def spectral_update(prm, fields7, x, y, z, rho_old, dt, chi, nthreads=1):
    """Returns (new chi [np,nbins], nsub [np] int32, lost [np])."""
    keep, fa = _fields(fields7)
    x, px = _d(x); y, py = _d(y); z, pz = _d(z); rho_old, pr = _d(rho_old)
    chi = np.array(chi, dtype=np.float64)
    n = x.shape[0]
    assert chi.shape == (n, prm.nbins)
    nsub = np.empty(n, dtype=np.int32); lost = np.empty(n)
    lib().orc_spectral_update(C.byref(prm), fa, C.c_int64(n), px, py, pz, pr, C.c_double(dt),
                              chi.ctypes.data_as(C.POINTER(C.c_double)),
                              nsub.ctypes.data_as(C.POINTER(C.c_int32)),
                              lost.ctypes.data_as(C.POINTER(C.c_double)), C.c_int32(nthreads))
    return chi, nsub, lost


def step(prm, fields7, x, y, z, dt, chi, nthreads=1):
    """One frozen-field step.  Returns (x, y, z, chi, nsub, lost, status), all new arrays."""
    keep, fa = _fields(fields7)
    x = np.array(x, dtype=np.float64); y = np.array(y, dtype=np.float64); z = np.array(z, dtype=np.float64)
    chi = np.array(chi, dtype=np.float64)
    n = x.shape[0]
    assert chi.shape == (n, prm.nbins)
    nsub = np.empty(n, dtype=np.int32); lost = np.empty(n); status = np.zeros(n, dtype=np.int32)
    dp = lambda a: a.ctypes.data_as(C.POINTER(C.c_double))
    lib().orc_step(C.byref(prm), fa, C.c_int64(n), dp(x), dp(y), dp(z), C.c_double(dt), dp(chi),
                   nsub.ctypes.data_as(C.POINTER(C.c_int32)), dp(lost),
                   status.ctypes.data_as(C.POINTER(C.c_int32)), C.c_int32(nthreads))
    return x, y, z, chi, nsub, lost, status
