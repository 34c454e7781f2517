"""lp_number_static, the one entry point of the library that allocates nothing, against the existing path.

Why the entry point exists (include/lp.h has the contract): some users of the LP kernels cannot call cudaMalloc
when they want the particle number of a set of spectra -- a conservation monitor inside a host code that owns all
device memory through its own arena, a diagnostic fired while other streams are running (an allocation would
stall the whole GPU), code placed where the allocating runtime calls are not allowed.  The existing way to get that
number, lp_get_diag, needs a context (lp_create allocates a table) and the workspace of the whole step.  The new
call keeps its partial sums in a 64 KiB array built into liblp_b200.so instead, which caps it at 2^24 rows.

What is checked: the number it writes equals lp_get_diag's number for the same spectra within the 1e-12 relative
bound the other tests put on aggregate sums (tests/test_gpu_parity.py::test_number_conservation_diag; the two
paths add in different orders), on two calls in a row that share the built-in scratch -- a large set first, a
small one second, so that partial sums left behind by the first call would show up in the second if they were
read -- then that a repeated call returns the same bits, that the device's free memory does not move across a call,
and that sizes beyond the limit are refused with a reason instead of overrunning the array.

This file is named to be collected last: `pytest -x` stops at the first failure, and a failure of this add-on must
not hide the parity tests.  It passes alone in a fresh process and after the other tests."""

import pytest
import torch

import lp_inputs as I
import paper_2602_23434_b200 as P

pytestmark = pytest.mark.gpu
B = P.binding

AGGREGATE_TOL = 1e-12        # as test_number_conservation_diag


def existing_path_number(w):
    """Spectra of workload w on the GPU and their number through lp_create / workspace / lp_get_diag."""
    fields = I.make_fields(w, device="cpu")
    x, y, z, pid = I.make_particles(w)
    chi = I.make_spectrum(w, jitter=True)
    lp = P.LP(P.config_from_workload(w, u_rad=0.0))
    lp.set_fields(fields)
    lp.bind_particles(x, y, z, pid, chi)
    number = lp.diag()["number"]
    _, widths = B.lp_get_bins(lp.ctx, w.nbins)
    chi_dev = lp.chi.clone()
    lp.close()
    return chi_dev, torch.as_tensor(widths).cuda(), number


def number_static(chi_dev, widths_dev, out):
    np_, nbins = chi_dev.shape
    B.lp_number_static(chi_dev.device.index, chi_dev.data_ptr(), widths_dev.data_ptr(), nbins, np_, out.data_ptr(),
                       torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    return float(out.item())


def test_number_static_matches_lp_get_diag_on_two_calls_in_a_row():
    big = I.workload(3).scaled(n=12, np=70001, nbins=64, sort_every=0)       # 35 tiles of 2048 rows, ragged tail
    small = I.workload(3).scaled(n=12, np=5000 + 3, nbins=128, sort_every=0, seed=11)   # 3 tiles
    chi_a, wid_a, want_a = existing_path_number(big)
    chi_b, wid_b, want_b = existing_path_number(small)
    out = torch.full((1,), float("nan"), dtype=torch.float64, device="cuda")

    got_a = number_static(chi_a, wid_a, out)             # first call on this device: also looks the scratch up
    free_before = torch.cuda.mem_get_info()[0]
    got_b = number_static(chi_b, wid_b, out)             # second call, on top of the first one's partial sums
    free_after = torch.cuda.mem_get_info()[0]
    assert want_a > 0 and want_b > 0
    assert abs(got_a / want_a - 1) < AGGREGATE_TOL, (got_a, want_a)
    assert abs(got_b / want_b - 1) < AGGREGATE_TOL, (got_b, want_b)
    assert free_after == free_before, "a call of lp_number_static changed the device's free memory"

    # the order of the additions depends on the sizes alone: the same input gives the same bits, whatever ran before
    assert number_static(chi_a, wid_a, out) == got_a
    assert number_static(chi_b, wid_b, out) == got_b
    # and against plain fp64 on the host, to rounding of a sum of positive terms
    ref = float((chi_b.cpu().numpy() @ wid_b.cpu().numpy()).sum())
    assert abs(got_b / ref - 1) < AGGREGATE_TOL


def test_number_static_edges_and_limits():
    wid = torch.ones(16, dtype=torch.float64, device="cuda")
    chi = torch.arange(3 * 16, dtype=torch.float64, device="cuda").reshape(3, 16)
    out = torch.full((1,), float("nan"), dtype=torch.float64, device="cuda")
    assert number_static(chi, wid, out) == float(sum(range(48)))             # small integers: exact
    assert number_static(chi[:0], wid, out) == 0.0                           # no rows: zero, no launch
    with pytest.raises(B.LPError) as e:                                      # one row past the built-in scratch
        B.lp_number_static(0, chi.data_ptr(), wid.data_ptr(), 16, (1 << 24) + 1, out.data_ptr(), None)
    assert e.value.status == B.LP_ERR_UNSUPPORTED and "16777216" in str(e.value)
    with pytest.raises(B.LPError) as e:
        B.lp_number_static(0, chi.data_ptr(), wid.data_ptr(), 513, 3, out.data_ptr(), None)
    assert e.value.status == B.LP_ERR_UNSUPPORTED and "nbins" in str(e.value)
    with pytest.raises(B.LPError) as e:
        B.lp_number_static(0, chi.data_ptr(), wid.data_ptr(), 16, 3, None, None)
    assert e.value.status == B.LP_ERR_INVALID_ARG
    assert number_static(chi, wid, out) == float(sum(range(48)))             # refusals left nothing behind
