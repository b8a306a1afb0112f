"""-m gpu: amr_conserved_totals_noalloc - the conserved-totals reduction for callers that cannot allocate (scratch in a
static device array, result written to a device array, nothing but a memset and a launch enqueued) - against the existing
path amr_conserved_totals on the same device data, on calls in a row that share the scratch array.  Collected last on
purpose (the suite runs with pytest -x); passes alone in a fresh process and after the other tests."""
import numpy as np
import pytest

import workloads as wk

pytestmark = pytest.mark.gpu

# the bound the conservation tests use for fp64 totals (north_star: "conserved totals agreeing to 1e-13"), relative to
# sum |U|: both paths add the same 256 per-block double sums, only the last sum differs (host long double / device tree)
TOL = 1e-13


def _batch(level, dtype):
    import paper_1412_0934_b200 as amr
    b = amr.PatchBatch.from_level(level, dtype)
    return b


def _both(b, nf, ncells, out):
    """(existing path, new entry point) on the batch's current device state; `out` is a device tensor the caller owns."""
    import torch
    import paper_1412_0934_b200 as amr
    ref = b.conserved_totals()
    out.fill_(float("nan"))
    amr.conserved_totals_noalloc(b.state_ptr(0), nf, ncells, ncells, out, dtype=b.dtype)
    torch.cuda.synchronize()
    absn = np.abs(b.download().astype(np.float64)).sum(axis=(1, 2, 3, 4))     # sum |U| of the state that was summed
    return ref, out[:nf].cpu().numpy(), absn


@pytest.mark.parametrize("np_dtype", [np.float64, np.float32])
def test_no_alloc_totals_match_the_existing_path_on_calls_in_a_row(np_dtype):
    import torch
    import paper_1412_0934_b200 as amr
    dtype = amr.AMR_F64 if np_dtype == np.float64 else amr.AMR_F32
    mhd = wk.config3_orszag_tang(N=64, n=16).levels[0]            # 9 fields, 64 patches of 16^3
    hyd = wk.config2_random_patches(npatch=48).levels[0]          # 5 fields, 48 patches of 16^3
    bm, bh = _batch(mhd, dtype), _batch(hyd, dtype)
    out = torch.empty(16, dtype=torch.float64, device="cuda")
    # call 1: nine fields; call 2: five fields of another batch (the scratch array still holds call 1's partial sums);
    # call 3: the nine fields again after a step has changed them; call 4: the same state once more (same bits)
    calls = []
    calls.append((mhd, _both(bm, 9, mhd.ncells, out)))
    calls.append((hyd, _both(bh, 5, hyd.ncells, out)))
    dt, sm = bm.cfl_dt(5.0 / 3.0, 0.3)
    bm.mhd_step(dt, 5.0 / 3.0, amr.AMR_LIM_MC, amr.AMR_RS_HLLD, sm, 0.4)
    free_before = torch.cuda.mem_get_info()[0]
    calls.append((mhd, _both(bm, 9, mhd.ncells, out)))
    calls.append((mhd, _both(bm, 9, mhd.ncells, out)))
    free_after = torch.cuda.mem_get_info()[0]
    assert free_after == free_before, "device memory in use changed across two calls"
    for lev, (ref, got, absn) in calls:
        assert np.isfinite(got).all()
        assert (np.abs(got - ref) <= TOL * absn).all(), (got, ref, absn)     # a field that is identically zero: 0 <= 0
    assert np.array_equal(calls[2][1][1], calls[3][1][1])
    # a sub-range and a stride: the first 7 patches of every field
    n7 = 7 * 16 ** 3
    out.fill_(float("nan"))
    amr.conserved_totals_noalloc(bm.state_ptr(0), 9, n7, mhd.ncells, out, dtype=dtype)
    torch.cuda.synchronize()
    ref7 = bm.download()[:, :7].astype(np.float64).sum(axis=(1, 2, 3, 4))
    absn7 = np.abs(bm.download()[:, :7].astype(np.float64)).sum(axis=(1, 2, 3, 4))
    assert (np.abs(out[:9].cpu().numpy() - ref7) <= 1e-12 * absn7).all()


def test_no_alloc_entry_point_rejects_what_it_cannot_hold():
    import torch
    import paper_1412_0934_b200 as amr
    u = torch.ones(17 * 1024, dtype=torch.float32, device="cuda")
    out = torch.zeros(17, dtype=torch.float64, device="cuda")
    with pytest.raises(amr.AmrError, match="AMR_NOALLOC_MAX_FIELDS"):
        amr.conserved_totals_noalloc(u, 17, 1024, 1024, out)                      # more fields than the static array fits
    with pytest.raises(amr.AmrError):
        amr.conserved_totals_noalloc(u, 4, 2048, 1024, out)                       # ncells > field_stride
    with pytest.raises(amr.AmrError):
        amr.conserved_totals_noalloc(u, 0, 1024, 1024, out)
    host = np.zeros(16)
    with pytest.raises(amr.AmrError):
        amr.conserved_totals_noalloc(u, 4, 1024, 1024, host.ctypes.data)          # the result must go to device memory
    # the maximum itself is accepted, and the array is left usable after the rejected calls
    amr.conserved_totals_noalloc(u, 16, 1024, 1024, out)
    torch.cuda.synchronize()
    assert np.array_equal(out[:16].cpu().numpy(), np.full(16, 1024.0))
