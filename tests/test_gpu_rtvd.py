"""GPU parity of the directionally split relaxing-TVD update (hydro_rtvd_solve_*) against
oracle/rtvd_oracle.cpp, element by element, at the bars of tests/test_gpu_parity.py (S22 / S23)."""
import numpy as np
import pytest

from paper_1103_3373_b200 import workloads as wl
from tests.harness import run_grid
from tests.test_gpu_parity import B, check  # noqa: F401  (B is a fixture)
from tests.test_oracle_rtvd import RtvdBackend

pytestmark = pytest.mark.gpu


def gpu_rtvd(B, G, dt, dh, gamma, order, **kw):
    import torch
    t = torch.from_numpy(np.ascontiguousarray(G)).cuda()
    status = torch.zeros(3, dtype=torch.int64, device="cuda")
    out, ff = B.hydro_rtvd_solve(t, dt, dh, gamma, order, status=status, **kw)
    torch.cuda.synchronize()
    return out.cpu().numpy(), (ff.cpu().numpy() if ff is not None else None), status.cpu().numpy()


@pytest.mark.parametrize("dtype", (np.float64, np.float32))
@pytest.mark.parametrize("order", (0, 1))
@pytest.mark.parametrize("Ng,g", ((5, 3), (1221, 3), (7, 5)))
def test_rtvd_matches_oracle(B, oracle, nthreads, dtype, order, Ng, g):
    gamma = 5.0 / 3.0
    G = wl.amr_batch(Ng, g=g, gamma=gamma, seed=31, dtype=np.dtype(dtype).name).numpy()
    dt = 0.3 / oracle.hydro_dt(G, gamma, 0)
    ref_out, ref_ff, ref_st = oracle.rtvd_solve(G, dt, 1.0, gamma, order=order, nthreads=nthreads)
    out, ff, st = gpu_rtvd(B, G, dt, 1.0, gamma, order)
    check(out, ff, ref_out, ref_ff, dtype, ("rtvd", order, Ng, g))
    assert st[1] == 0 and ref_st[1] == 0


def test_rtvd_uniform_bitwise_edge_cases_and_errors(B):
    import torch
    G = torch.empty((3, 5, 22, 22, 22), dtype=torch.float64, device="cuda")
    for q, v in enumerate((1.3, 0.4, -0.7, 0.2, 2.9)):
        G[:, q] = v
    out, ff = B.hydro_rtvd_solve(G, 0.05, 1.0, 1.4, 0)
    assert torch.equal(out, G[:, :, 3:19, 3:19, 3:19])
    # no groups: a no-op; face fluxes off; a bad state is counted
    B.hydro_rtvd_solve(G[:0], 0.05, 1.0, 1.4, 0)
    assert B.hydro_rtvd_solve(G, 0.05, 1.0, 1.4, 1, face_flux=False)[1] is None
    bad = G.clone()
    bad[1, 4, 10, 10, 10] = -1.0
    st = torch.zeros(3, dtype=torch.int64, device="cuda")
    B.hydro_rtvd_solve(bad, 0.05, 1.0, 1.4, 0, status=st)
    assert st.cpu().tolist()[1] > 0
    with pytest.raises(B.HydroError):
        B.hydro_rtvd_solve(torch.ones((1, 5, 20, 20, 20), dtype=torch.float64, device="cuda"), 0.05, 1.0, 1.4, 0)  # g = 2 < 3
    with pytest.raises(B.HydroError):
        B.hydro_rtvd_solve(G, 0.05, 1.0, 1.4, 2)
    with pytest.raises(B.HydroError):
        B.hydro_rtvd_solve(G, 0.05, 1.0, 1.4, 0, workspace=torch.empty(1024, dtype=torch.uint8, device="cuda"))


class CudaRtvd:
    def __init__(self, B):
        self.B, self.step = B, 0

    def dt(self, G, gamma, norm):
        import torch
        return float(self.B.hydro_dt(torch.from_numpy(np.ascontiguousarray(G)).cuda(), gamma, norm).item())

    def solve(self, G, dt, dh, gamma, scheme, riemann, limiter, **kw):
        order = self.step & 1
        self.step += 1
        return gpu_rtvd(self.B, G, dt, dh, gamma, order)


@pytest.mark.parametrize("dtype", (np.float64, np.float32))
def test_rtvd_multi_step_blast(B, oracle, nthreads, dtype):
    # the config-2 workload shape (blast, periodic) through alternating sweep orders, 10 steps, against the oracle
    gamma, N, steps = 5.0 / 3.0, 32, 10
    U0 = wl.blast_grid(N, radius=3.0, gamma=gamma, p_ambient=1e-2, dtype=dtype)
    Ur, _, _, _ = run_grid(RtvdBackend(oracle, nthreads), U0.copy(), steps, 1.0, gamma, 3, 0, 0, cfl=0.4, g=3)
    Ug, _, st, _ = run_grid(CudaRtvd(B), U0.copy(), steps, 1.0, gamma, 3, 0, 0, cfl=0.4, g=3)
    from tests.test_gpu_parity import err_l1, err_max
    if dtype == np.float64:
        assert err_max(Ug[None], Ur[None]) <= 1e-12
    else:
        assert err_l1(Ug[None], Ur[None]) <= steps * 1e-5
    assert st[1] == 0
    for v in (0, 4):
        assert abs(Ug[v].sum(dtype=np.float64) - U0[v].sum(dtype=np.float64)) <= (1e-6 if dtype == np.float32 else 1e-13) * U0[v].sum(dtype=np.float64)
