"""CPU-side checks of the boundary: the library builds, loads and exports every symbol that
include/lp.h declares; argument validation that needs no GPU; binding struct layout."""
import ctypes as C
import os
import re

import pytest

import paper_2602_23434_b200 as P

B = P.binding
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "lp.h")).read()
    return sorted(set(re.findall(r"LP_API\s+[\w\s\*]+?\b(lp_\w+)\s*\(", src)))


def test_library_exports_every_declared_symbol():
    lib = B.load()
    names = declared_symbols()
    assert len(names) >= 32 and set(names) == set(B.EXPORTS)
    for n in names:
        assert getattr(lib, n) is not None


def test_struct_sizes_match_the_header():
    # compile a tiny C program against include/lp.h and compare sizeof with the ctypes mirrors
    import subprocess, tempfile
    with tempfile.TemporaryDirectory() as d:
        c = os.path.join(d, "s.c")
        open(c, "w").write('#include <stdio.h>\n#include "lp.h"\nint main(){printf("%zu %zu\\n",'
                           'sizeof(lp_config),sizeof(lp_diag));return 0;}\n')
        exe = os.path.join(d, "s")
        subprocess.run(["gcc", "-I", os.path.join(ROOT, "include"), c, "-o", exe], check=True)
        a, b = subprocess.run([exe], capture_output=True, text=True, check=True).stdout.split()
    assert int(a) == C.sizeof(B.lp_config) and int(b) == C.sizeof(B.lp_diag)


def cfg(**kw):
    d = dict(nx=8, ny=8, nz=8, xlo=(-1,) * 3, xhi=(1,) * 3, periodic=(1, 1, 1), np=100, nbins=64,
             e_min=1.0, e_max=1e6)
    d.update(kw)
    return P.make_config(**d)


@pytest.mark.parametrize("bad,status", [
    (dict(nbins=48), B.LP_ERR_UNSUPPORTED),
    (dict(nbins=1024), B.LP_ERR_UNSUPPORTED),
    (dict(nx=0), B.LP_ERR_INVALID_ARG),
    (dict(nx=2048, ny=2048, nz=2048), B.LP_ERR_UNSUPPORTED),
    (dict(e_min=0.0), B.LP_ERR_INVALID_ARG),
    (dict(e_max=0.5), B.LP_ERR_INVALID_ARG),
    (dict(cfl_e=1.5), B.LP_ERR_INVALID_ARG),
    (dict(max_substeps=0), B.LP_ERR_INVALID_ARG),
    (dict(np=-1), B.LP_ERR_INVALID_ARG),
    (dict(xhi=(1, -1, 1)), B.LP_ERR_INVALID_ARG),
])
def test_config_validation_without_gpu(bad, status):
    with pytest.raises(B.LPError) as e:
        B.lp_workspace_bytes(cfg(**bad))
    assert e.value.status == status


def test_struct_size_is_checked():
    c = cfg()
    c.struct_size = 8
    with pytest.raises(B.LPError) as e:
        B.lp_workspace_bytes(c)
    assert e.value.status == B.LP_ERR_INVALID_ARG


def test_workspace_bytes_grow_with_problem():
    a = B.lp_workspace_bytes(cfg())
    b = B.lp_workspace_bytes(cfg(np=200))
    c = B.lp_workspace_bytes(cfg(nx=16))
    assert a % 256 == 0 and b > a and c > a
    # dominated by the alternate chi rows + cell records: np*nbins*8 + 64*ncell
    assert a >= 100 * 64 * 8 + 64 * 512


def test_null_arguments_are_rejected_not_crashed():
    lib = B.load()
    assert lib.lp_create(None, None) == B.LP_ERR_INVALID_ARG
    out = C.c_void_p()
    assert lib.lp_create(None, C.byref(out)) == B.LP_ERR_INVALID_ARG and not out
    assert lib.lp_destroy(None) == B.LP_ERR_INVALID_ARG
    assert lib.lp_step(None, 0.1, None) == B.LP_ERR_INVALID_ARG
    assert lib.lp_last_error(None) == b"null context"


def test_product_path_has_no_cpu_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(RuntimeError):
        P.LP(cfg())


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2602_23434_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src and "lp_oracle" not in src, f


@pytest.mark.parametrize("nbins,e_min,e_max", [(16, 1.0, 1e8), (64, 1e1, 1e6), (64, 1.0, 1e8), (128, 1.0, 1e7),
                                                (256, 1.0, 1e8), (512, 1.0, 1e8), (32, 0.5, 3.0)])
def test_cfl_candidate_bins_carry_the_maximum(nbins, e_min, e_max):
    """Host logic of step a8: lp_create reduces the CFL max over bins to the hull-vertex bins.
    Brute force over all bins (plain numpy fp64, the oracle's formula) must give the same lambda for
    any (a, c_r >= 0) up to the rounding of one evaluation."""
    import numpy as np
    lib = B.load()
    c = cfg(nbins=nbins, e_min=e_min, e_max=e_max)
    ctx = C.c_void_p()
    st = lib.lp_create(C.byref(c), C.byref(ctx))      # no GPU here: LP_ERR_CUDA, but the context exists
    assert ctx and st in (B.LP_OK, B.LP_ERR_CUDA)
    try:
        cand = B.lp_get_cfl_bins(ctx)
        E, dE = B.lp_get_bins(ctx, nbins)
    finally:
        lib.lp_destroy(ctx)
    assert cand is not None and 0 in cand and nbins - 1 in cand and len(cand) <= 24
    rng = np.random.default_rng(nbins)
    cases = [(a, cr) for a in (-3.0, -1e-3, 0.0, 1e-3, 2.0) for cr in (0.0, 1e-9, 1e-6, 1e-3)]
    cases += [(float(rng.normal() * 10 ** rng.uniform(-4, 2)), float(10 ** rng.uniform(-12, -2))) for _ in range(400)]
    # sign change of w placed inside the table: a = -c_r * E_k
    cases += [(-1e-6 * float(E[k]) * (1 + 1e-9), 1e-6) for k in range(0, nbins + 1, max(1, nbins // 16))]
    for a, cr in cases:
        w = -E * (a + cr * E)
        out = (np.maximum(w[1:], 0.0) - np.minimum(w[:-1], 0.0)) / dE
        lam_all = out.max()
        lam_cand = out[cand].max()
        assert lam_all <= lam_cand * (1 + 1e-15), (a, cr, int(out.argmax()), cand)


@pytest.mark.parametrize("n,e,cap", [(0, 18, 0), (1, 18, 262144), (262144, 18, 262144), (262145, 18, 524288),
                                     (16777216, 18, 16777216), (1000, 4, 1008), (1024, 4, 1024)])
def test_chunked_capacity_is_listing_1(n, e, cap):
    """Listing 1: N_c = (N >> e) + (N % L == 0 ? 0 : 1) chunks of L = 2^e."""
    assert B.lp_chunked_capacity(n, e) == cap
    assert cap % (1 << e) == 0 and cap >= n and cap - n < (1 << e)


def test_set_count_stays_within_capacity():
    lib = B.load()
    c = cfg()
    ctx = C.c_void_p()
    st = lib.lp_create(C.byref(c), C.byref(ctx))
    assert ctx and st in (B.LP_OK, B.LP_ERR_CUDA)
    try:
        assert lib.lp_set_count(ctx, C.c_int64(c.np + 1)) == B.LP_ERR_INVALID_ARG
        assert lib.lp_set_count(ctx, C.c_int64(-1)) == B.LP_ERR_INVALID_ARG
        assert lib.lp_set_count(ctx, C.c_int64(0)) == B.LP_OK
    finally:
        lib.lp_destroy(ctx)


def test_number_static_refuses_oversize_without_touching_the_gpu():
    """lp_number_static (the allocation-free entry point) checks its sizes before any CUDA call: the refusal and
    its reason can be had on a box without a GPU."""
    with pytest.raises(B.LPError) as e:
        B.lp_number_static(0, 8, 8, 64, (1 << 24) + 1, 8, None)
    assert e.value.status == B.LP_ERR_UNSUPPORTED and "static scratch" in str(e.value)
    with pytest.raises(B.LPError) as e:
        B.lp_number_static(0, 8, 8, 0, 10, 8, None)
    assert e.value.status == B.LP_ERR_UNSUPPORTED
    with pytest.raises(B.LPError) as e:
        B.lp_number_static(-1, 8, 8, 64, 10, 8, None)
    assert e.value.status == B.LP_ERR_INVALID_ARG
