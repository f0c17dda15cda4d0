"""hz_sum_fields_noalloc (include/hz.h; csrc/hz_noalloc.cu): the one entry point that allocates nothing, for callers
that cannot call cudaMalloc.  Its sums must agree with the existing path -- hz_diagnostics' conservation sums
(k_diag + k_diag_final, scratch inside the context) -- within the 1e-12 the diagnostics tests use for sums
(summation order differs, R21), on two calls in a row that share the fixed scratch array.

The file name sorts after every other test file on purpose: the suite runs with pytest -x, and a failure here
must not hide the tests of the hot path.  It needs nothing from them: it passes alone in a fresh process too."""
import numpy as np
import pytest

import workloads as wl

pytestmark = pytest.mark.gpu

SUM_KEYS = ("sumD", "sumSx", "sumSy", "sumSz", "sumTau", "sumBx", "sumBy", "sumBz", "sumPsi")


def _check(hz, w, dtype):
    """One call of the new entry point on the context's conserved fields against hz_diagnostics."""
    import torch
    from paper_1102_5202_b200 import binding as B
    td = torch.float64 if dtype == "f64" else torch.float32
    cons = torch.empty((9,) + w.alpha.shape, dtype=td, device="cuda")
    hz.get_conserved(out=cons)                                   # the input: 9 planes of ncell elements, device
    out = torch.full((9,), float("nan"), dtype=torch.float64, device="cuda")
    B.sum_fields_noalloc(cons, 9, w.ncell, out)
    torch.cuda.synchronize()
    dV = w.h[0] * w.h[1] * w.h[2]
    got = out.cpu().numpy() * dV
    ref = hz.diagnostics()
    # 1e-12 as in test_diagnostics_match_oracle (floor 1e-3), measured against the size of what is summed: a sum
    # that cancels by symmetry (the momentum of a periodic wave) has no scale of its own
    l1 = cons.double().abs().reshape(9, -1).sum(dim=1).cpu().numpy() * dV
    plain = cons.double().reshape(9, -1).sum(dim=1).cpu().numpy() * dV      # a plain fp64 sum of the same array
    for i, k in enumerate(SUM_KEYS):
        tol = 1e-12 * max(abs(ref[k]), l1[i], 1e-3)
        assert abs(got[i] - ref[k]) <= tol, (dtype, k, got[i], ref[k])
        assert abs(got[i] - plain[i]) <= tol, (dtype, k, got[i], plain[i])
    return got


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_two_calls_in_a_row_match_the_diagnostics_path(dtype):
    """First call: 48^3 cells (432 blocks of partials).  Second call, straight after it: a 20 x 12 x 9 grid (9 blocks),
    after a Runge-Kutta step, so stale rows of the first call lie beyond it in the shared scratch array and the
    cleaning scalar (sumPsi) is no longer zero.  Then the first grid once more."""
    from paper_1102_5202_b200 import Horizon
    from paper_1102_5202_b200 import binding as B
    B.noalloc_setup()
    big, small = wl.kerr_sweep(48), wl.alfven_wave(n=(20, 12, 9))
    a = Horizon.from_workload(big, dtype=dtype)
    b = Horizon.from_workload(small, dtype=dtype)
    b.step(small.dt, 1)
    s1 = _check(a, big, dtype)
    s2 = _check(b, small, dtype)
    s3 = _check(a, big, dtype)
    assert np.array_equal(s1, s3)          # deterministic: fixed summation order, no leftovers from call 2
    assert not np.allclose(s1[:5], s2[:5])
    a.close(); b.close()


def test_it_allocates_nothing_and_refuses_sizes_beyond_the_scratch():
    import torch
    from paper_1102_5202_b200 import binding as B
    x = torch.rand((16, 1000), dtype=torch.float64, device="cuda")
    out = torch.empty(16, dtype=torch.float64, device="cuda")
    B.sum_fields_noalloc(x, 16, 1000, out)                       # the most fields one call takes
    torch.cuda.synchronize()
    assert torch.allclose(out, x.sum(dim=1), rtol=1e-13)
    # a repeat call (kernels loaded, scratch address known) leaves the device's free memory where it was
    free0 = torch.cuda.mem_get_info()[0]
    for _ in range(3):
        B.sum_fields_noalloc(x, 16, 1000, out)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0
    y = torch.empty(17 * 8, dtype=torch.float64, device="cuda")
    with pytest.raises(B.HzError) as e:
        B.sum_fields_noalloc(y, 17, 8, out)                      # more fields than a row of the scratch holds
    assert e.value.code == B.HZ_ELIMIT and "maximum" in str(e.value)
    with pytest.raises(B.HzError) as e:
        B.sum_fields_noalloc(x, 1, B.HZ_NOALLOC_MAX_CELLS + 1, out)
    assert e.value.code == B.HZ_ELIMIT
    with pytest.raises(B.HzError) as e:
        B.sum_fields_noalloc(x.cpu(), 16, 1000, out)             # host memory is not accepted
    assert e.value.code == B.HZ_EINVAL
    # a non-default stream, ordered by the caller
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(s):
        B.sum_fields_noalloc(x, 16, 1000, out, stream=s)
    s.synchronize()
    assert torch.allclose(out, x.sum(dim=1), rtol=1e-13)
