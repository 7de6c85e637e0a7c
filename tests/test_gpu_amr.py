"""GPU parity for the consumer of face_flux (hydro_fluxfix_*, hydro_restrict_*, hydro_flux_accum_*):
against oracle/amr_oracle.cpp element by element -- bit-exact where every cell receives one contribution (the index
plumbing and the rounding sequence are the oracle's), to rounding where several faces meet in one cell (atomic order) --
and through the property that pins the whole construction: two-level conservation with the fluxes of the CUDA solver.
"""
import numpy as np
import pytest

from tests.harness import CudaBackend, OracleBackend, two_level_lists, two_level_step
from tests.test_oracle_amr import ORIGINS, composite

pytestmark = pytest.mark.gpu

MHM, VL, CTU = 0, 1, 2
HLLE, HLLC, ROE = 1, 2, 3


@pytest.fixture(scope="module")
def B():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("gpu tests need a CUDA device")
    from paper_1103_3373_b200 import binding
    binding.lib()
    return binding


class CudaAmr:
    """numpy in / numpy out adapter of the three CUDA entry points (in place on the numpy array, like the oracle's)."""

    def __init__(self, B):
        import torch
        self.B, self.torch = B, torch

    def _d(self, a):
        return self.torch.from_numpy(np.ascontiguousarray(a)).cuda()

    def restrict(self, fine_out, coarse_out, rmap):
        c = self._d(coarse_out)
        self.B.hydro_restrict(self._d(fine_out), c, self._d(np.asarray(rmap, np.int32)))
        coarse_out[...] = c.cpu().numpy()
        return coarse_out

    def fluxfix(self, coarse_out, coarse_flux, fine_flux, faces, dt_c, dh_c):
        c = self._d(coarse_out)
        self.B.hydro_fluxfix(c, self._d(coarse_flux), self._d(fine_flux), self._d(np.asarray(faces, np.int32)), dt_c, dh_c)
        coarse_out[...] = c.cpu().numpy()
        return coarse_out


@pytest.mark.parametrize("dtype", (np.float64, np.float32))
def test_fluxfix_restrict_bit_exact_on_random_data(B, oracle, dtype):
    rng = np.random.default_rng(5)
    Nc, Nf = 8, 3
    co = rng.normal(size=(Nc, 5, 16, 16, 16)).astype(dtype)
    cf = rng.normal(size=(Nc, 9, 5, 16, 16)).astype(dtype)
    ff = rng.normal(size=(Nf, 9, 5, 16, 16)).astype(dtype)
    fo = rng.normal(size=(Nf, 5, 16, 16, 16)).astype(dtype)
    # three refined patches of a 32^3 coarse grid, far enough apart that no coarse cell gets two contributions
    faces, rmap = [], []
    for n, origin in enumerate(ORIGINS):
        f, r = two_level_lists(origin, 32)
        f[:, 0] = n
        r[:, 0] = n
        faces.append(f)
        rmap.append(r)
    faces, rmap = np.concatenate(faces), np.concatenate(rmap)
    ref = co.copy()
    oracle.restrict(fo, ref, rmap)
    oracle.fluxfix(ref, cf, ff, faces, dtype(0.01), dtype(0.03125))
    got = co.copy()
    amr = CudaAmr(B)
    amr.restrict(fo, got, rmap)
    amr.fluxfix(got, cf, ff, faces, 0.01, 0.03125)
    assert np.array_equal(got, ref)
    assert not np.array_equal(got, co)


def test_fluxfix_meeting_faces_and_edge_cases(B, oracle):
    import torch
    # two entries that correct the SAME coarse cells (a cell with refined neighbours on two sides): order-free to rounding
    rng = np.random.default_rng(6)
    co = rng.normal(size=(1, 5, 16, 16, 16))
    cf = rng.normal(size=(1, 9, 5, 16, 16))
    ff = rng.normal(size=(2, 9, 5, 16, 16))
    faces = np.array([[0, 0, 0, 0, 7, 0, 0], [1, 0, 1, 0, 7, 0, 0]], np.int32)  # layer i = 7 corrected from above and from below
    ref = co.copy()
    oracle.fluxfix(ref, cf, ff, faces, 0.02, 0.5)
    got = CudaAmr(B).fluxfix(co.copy(), cf, ff, faces, 0.02, 0.5)
    assert np.allclose(got, ref, rtol=0, atol=4e-16 * np.abs(ref).max())
    # empty lists are no-ops; null pointers and negative counts are argument errors
    t = torch.zeros((1, 5, 16, 16, 16), dtype=torch.float64, device="cuda")
    f9 = torch.zeros((1, 9, 5, 16, 16), dtype=torch.float64, device="cuda")
    empty = torch.zeros((0, 7), dtype=torch.int32, device="cuda")
    B.hydro_fluxfix(t, f9, f9, empty, 0.1, 1.0)
    B.hydro_restrict(t, t, torch.zeros((0, 5), dtype=torch.int32, device="cuda"))
    L = B.lib()
    one = torch.zeros((1, 7), dtype=torch.int32, device="cuda")
    assert L.hydro_fluxfix_f64(None, f9.data_ptr(), f9.data_ptr(), one.data_ptr(), 1, 0.1, 1.0, None) == -3
    assert L.hydro_fluxfix_f64(t.data_ptr(), f9.data_ptr(), f9.data_ptr(), one.data_ptr(), -1, 0.1, 1.0, None) == -2
    assert L.hydro_fluxfix_f64(t.data_ptr(), f9.data_ptr(), f9.data_ptr(), one.data_ptr(), 1, 0.1, 0.0, None) == -7
    assert L.hydro_restrict_f64(t.data_ptr(), None, one.data_ptr(), 1, None) == -3


@pytest.mark.parametrize("dtype", (np.float64, np.float32))
def test_flux_accum_matches_oracle(B, oracle, dtype):
    import torch
    rng = np.random.default_rng(7)
    acc = rng.normal(size=(3, 9, 5, 16, 16)).astype(dtype)
    ff = rng.normal(size=(3, 9, 5, 16, 16)).astype(dtype)
    ref = oracle.flux_accum(acc.copy(), ff, dtype(0.5))
    a = torch.from_numpy(acc).cuda()
    B.hydro_flux_accum(a, torch.from_numpy(ff).cuda(), 0.5)
    assert np.array_equal(a.cpu().numpy(), ref)


@pytest.mark.parametrize("origin", ORIGINS)
@pytest.mark.parametrize("scheme,riemann", ((CTU, ROE), (MHM, HLLC)))
def test_two_level_step_on_the_gpu(B, oracle, nthreads, origin, scheme, riemann):
    # the whole two-level step on the device (hydro_solve fused kernels -> hydro_restrict -> hydro_fluxfix): conservative
    # to summation rounding, and equal to the all-oracle step within the fp64 parity bar
    gamma = 1.4
    Uc, Uf, dh = composite(origin)
    dt = 0.2 * (dh / 2) / 3.0
    new_gpu, fine_gpu = two_level_step(CudaBackend(2), CudaAmr(B), Uc, Uf, origin, dt, dh, gamma, scheme, riemann, 1)
    new_ref, fine_ref = two_level_step(OracleBackend(oracle, nthreads), oracle, Uc, Uf, origin, dt, dh, gamma, scheme, riemann, 1)
    tot0 = Uc.sum(axis=(1, 2, 3), dtype=np.float64)
    drift = np.abs(new_gpu.sum(axis=(1, 2, 3), dtype=np.float64) - tot0) / np.abs(Uc).sum(axis=(1, 2, 3))
    assert drift.max() < 2e-15, drift
    for q in range(5):
        sc = np.abs(new_ref[1:4]).max() if 1 <= q <= 3 else np.abs(new_ref[q]).max()
        assert np.abs(new_gpu[q] - new_ref[q]).max() <= 1e-12 * sc
