"""GPU parity of the directionally split weighted-average-flux update (hydro_waf_solve_*) against
oracle/waf_oracle.cpp, element by element, at the bars of tests/test_gpu_parity.py (S22 / S23)."""
import numpy as np
import pytest

from paper_1103_3373_b200 import workloads as wl
from tests.harness import run_grid
from tests.test_gpu_parity import B, check  # noqa: F401  (B is a fixture)
from tests.test_oracle_waf import WafBackend

pytestmark = pytest.mark.gpu


def gpu_waf(B, G, dt, dh, gamma, order, **kw):
    import torch
    t = torch.from_numpy(np.ascontiguousarray(G)).cuda()
    status = torch.zeros(3, dtype=torch.int64, device="cuda")
    out, ff = B.hydro_waf_solve(t, dt, dh, gamma, order, status=status, **kw)
    torch.cuda.synchronize()
    return out.cpu().numpy(), (ff.cpu().numpy() if ff is not None else None), status.cpu().numpy()


@pytest.mark.parametrize("dtype", (np.float64, np.float32))
@pytest.mark.parametrize("order", (0, 1))
@pytest.mark.parametrize("Ng,g", ((5, 3), (1221, 3), (7, 5)))
def test_waf_matches_oracle(B, oracle, nthreads, dtype, order, Ng, g):
    gamma = 5.0 / 3.0
    G = wl.amr_batch(Ng, g=g, gamma=gamma, seed=33, dtype=np.dtype(dtype).name).numpy()
    dt = 0.3 / oracle.hydro_dt(G, gamma, 0)
    ref_out, ref_ff, ref_st = oracle.waf_solve(G, dt, 1.0, gamma, order=order, nthreads=nthreads)
    out, ff, st = gpu_waf(B, G, dt, 1.0, gamma, order)
    check(out, ff, ref_out, ref_ff, dtype, ("waf", order, Ng, g))
    assert st[1] == 0 and ref_st[1] == 0


def test_waf_uniform_bitwise_and_edge_cases(B):
    import torch
    G = torch.empty((3, 5, 22, 22, 22), dtype=torch.float64, device="cuda")
    for q, v in enumerate((1.3, 0.4, -0.7, 0.2, 2.9)):
        G[:, q] = v
    for order in (0, 1):
        out, ff = B.hydro_waf_solve(G, 0.05, 1.0, 1.4, order)
        assert torch.equal(out, G[:, :, 3:19, 3:19, 3:19])
    Gf = G.float()
    out, _ = B.hydro_waf_solve(Gf, 0.05, 1.0, 1.4, 0)
    assert torch.equal(out, Gf[:, :, 3:19, 3:19, 3:19])
    empty = torch.empty((0, 5, 22, 22, 22), dtype=torch.float64, device="cuda")
    assert B.hydro_waf_solve(empty, 0.05, 1.0, 1.4, 0)[0].shape[0] == 0
    with pytest.raises(B.HydroError):
        B.hydro_waf_solve(G, 0.05, 1.0, 1.4, 2)
    with pytest.raises(B.HydroError):
        B.hydro_waf_solve(torch.empty((1, 5, 20, 20, 20), dtype=torch.float64, device="cuda"), 0.05, 1.0, 1.4, 0)


# a supersonic flow in both directions (all three waves of a face on one side), a strong shock: the upwind choices and the
# first-order limit of the limiter
@pytest.mark.parametrize("dtype", (np.float64, np.float32))
def test_waf_sod_and_supersonic_steps(B, oracle, nthreads, dtype):
    gamma = 1.4
    for vx in (0.0, 3.0, -3.0):
        U0 = np.ascontiguousarray(wl.sod_grid(32, axis=0, gamma=gamma)[:, :16, :16, :]).astype(dtype)
        rho = U0[0].copy()
        U0[4] += 0.5 * rho * vx * vx + U0[1] * vx   # Galilean boost along x
        U0[1] += rho * vx
        G = wl.grid_to_groups(U0, 3, "outflow")
        dt = 0.4 / 32 / oracle.hydro_dt(G, gamma, 0)
        for order in (0, 1):
            ref_out, ref_ff, _ = oracle.waf_solve(G, dt, 1.0 / 32, gamma, order=order, nthreads=nthreads)
            out, ff, st = gpu_waf(B, G, dt, 1.0 / 32, gamma, order)
            check(out, ff, ref_out, ref_ff, dtype, ("waf sod", vx, order))
