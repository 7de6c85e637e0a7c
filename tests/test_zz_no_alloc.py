"""hydro_rtvd_solve_noalloc_f64: the entry point that allocates nothing (scratch in a file-scope device array of the library)
against the existing path hydro_rtvd_solve_f64 (caller workspace), on two calls in a row.  Named test_zz_* so that pytest collects
it LAST: the suite runs with `pytest -x`, and a failure here must not hide the other tests.  Passes alone in a fresh process
and after the other tests (it depends on no state but the library)."""
import pytest

from paper_1103_3373_b200 import workloads as wl

pytestmark = pytest.mark.gpu
TOL64 = 1e-12  # the fp64 bar of tests/test_gpu_parity.py (S22); the two paths run the same kernel, so they agree bit for bit


@pytest.fixture(scope="module")
def B():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    from paper_1103_3373_b200 import binding
    binding.lib()
    return binding


def rel_err(got, ref):
    # S22: max |got - ref| / max |ref| per field, the three momenta pooled; got, ref [Ng, 5, 16, 16, 16]
    g, r = got.double(), ref.double()
    worst = 0.0
    for sl in (slice(0, 1), slice(1, 4), slice(4, 5)):
        worst = max(worst, (g[:, sl] - r[:, sl]).abs().max().item() / r[:, sl].abs().max().item())
    return worst


def rel_err_ff(got, ref):
    g, r = got.double(), ref.double()  # [Ng, 9, 5, 16, 16]
    worst = 0.0
    for sl in (slice(0, 1), slice(1, 4), slice(4, 5)):
        worst = max(worst, (g[:, :, sl] - r[:, :, sl]).abs().max().item() / r[:, :, sl].abs().max().item())
    return worst


def test_noalloc_matches_workspace_path_on_two_calls_in_a_row(B):
    import torch
    gamma = 5.0 / 3.0
    out_n = torch.empty((1500, 5, 16, 16, 16), dtype=torch.float64, device="cuda")
    ff_n = torch.empty((1500, 9, 5, 16, 16), dtype=torch.float64, device="cuda")
    # two calls in a row through the shared static scratch: different inputs, sizes (more and fewer groups than the 32 slots
    # would serve in one wave, and a ragged count) and sweep orders, so that stale contents of the first call would show
    for call, (Ng, seed, order) in enumerate(((1500, 41, 0), (37, 42, 1))):
        G = wl.amr_batch(Ng, g=3, gamma=gamma, seed=seed, dtype="float64").cuda()
        dt = 0.3 / float(B.hydro_dt(G, gamma, 0).item())
        st_ref = torch.zeros(3, dtype=torch.int64, device="cuda")
        st_n = torch.zeros(3, dtype=torch.int64, device="cuda")
        ref_out, ref_ff = B.hydro_rtvd_solve(G, dt, 1.0, gamma, order, status=st_ref)     # existing path: caller workspace
        out, ff = B.hydro_rtvd_solve_noalloc(G, dt, 1.0, gamma, order, out=out_n[:Ng], face_flux=ff_n[:Ng], status=st_n)
        torch.cuda.synchronize()
        assert torch.isfinite(out).all().item()
        assert rel_err(out, ref_out) <= TOL64, (call, rel_err(out, ref_out))
        assert rel_err_ff(ff, ref_ff) <= TOL64, call
        assert torch.equal(out, ref_out) and torch.equal(ff, ref_ff), call   # same kernel, independent groups: bitwise
        assert st_n.tolist() == st_ref.tolist()


def test_noalloc_limits_and_errors(B):
    import torch
    L = B.lib()
    big = B.RTVD_NOALLOC_MAX_GROUPS + 1
    a = 4096  # fake aligned "device" address: argument errors are detected on the host before any launch
    import ctypes as C
    f = lambda Ng, order=0, dt=0.1, gamma=1.4: L.hydro_rtvd_solve_noalloc_f64(a, 2 * a, None, Ng, C.c_double(dt), C.c_double(1.0),
                                                                            C.c_double(gamma), order, None, None)
    assert f(big) == -9 and "maximum" in B.hydro_strerror(-9)
    assert f(-1) == -2 and f(1, order=2) == -1 and f(1, dt=-1.0) == -7 and f(1, gamma=1.0) == -7
    assert f(0) == 0
    with pytest.raises(B.HydroError):
        G = torch.zeros((big, 5, 22, 22, 22), dtype=torch.float64, device="cuda")
        B.hydro_rtvd_solve_noalloc(G, 0.1, 1.0, 1.4, 0, out=torch.empty((big, 5, 16, 16, 16), dtype=torch.float64, device="cuda"))
