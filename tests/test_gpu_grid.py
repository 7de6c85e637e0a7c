"""SURVEY.md 8(f)-1 on the GPU: device-side gather / scatter for uniform grids (bit-exact against the numpy
definition in workloads.py, which the CUDA path does not use) and the on-device multi-step driver."""
import numpy as np
import pytest

from paper_1103_3373_b200 import workloads as wl
from tests.harness import CudaBackend, OracleBackend, run_grid

pytestmark = pytest.mark.gpu
CTU, ROE, HLLC, VANLEER = 2, 3, 2, 1


@pytest.fixture(scope="module")
def B():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    from paper_1103_3373_b200 import binding
    binding.lib()
    return binding


@pytest.mark.parametrize("dtype", (np.float32, np.float64))
@pytest.mark.parametrize("bc", ("periodic", "outflow"))
@pytest.mark.parametrize("g", (2, 3, 4))
def test_gather_scatter_bit_exact(B, dtype, bc, g):
    import torch
    rng = np.random.default_rng(g)
    U = rng.standard_normal((5, 32, 48, 16)).astype(dtype)   # Nz, Ny, Nx all different
    ref = wl.grid_to_groups(U, g, bc)
    Ud = torch.from_numpy(U).cuda()
    G = B.hydro_gather(Ud, g, B.BC_PERIODIC if bc == "periodic" else B.BC_OUTFLOW)
    assert np.array_equal(G.cpu().numpy(), ref)
    out = torch.from_numpy(np.ascontiguousarray(ref[:, :, g:g + 16, g:g + 16, g:g + 16])).cuda()
    back = B.hydro_scatter(out, U.shape[1:])
    assert np.array_equal(back.cpu().numpy(), U)
    assert np.array_equal(back.cpu().numpy(), wl.groups_to_grid(out.cpu().numpy(), U.shape[1:]))


# the gather kernel walks the groups in 4 x 4 x 4 bricks and the rest in plain order: a grid with full bricks AND a ragged
# remainder along every axis (6 x 9 x 5 groups), against the numpy definition
@pytest.mark.parametrize("dtype", (np.float32, np.float64))
@pytest.mark.parametrize("bc", ("periodic", "outflow"))
def test_gather_bricks_and_remainder_bit_exact(B, dtype, bc):
    import torch
    rng = np.random.default_rng(7)
    U = rng.standard_normal((5, 80, 144, 96)).astype(dtype)
    for g in (2, 3):
        ref = wl.grid_to_groups(U, g, bc)
        G = B.hydro_gather(torch.from_numpy(U).cuda(), g, B.BC_PERIODIC if bc == "periodic" else B.BC_OUTFLOW)
        assert np.array_equal(G.cpu().numpy(), ref)


def test_gather_argument_errors(B):
    import torch
    bad = torch.zeros((5, 16, 16, 24), device="cuda")
    with pytest.raises(B.HydroError):
        B.hydro_gather(bad, 2)
    ok = torch.zeros((5, 16, 16, 16), device="cuda")
    with pytest.raises(B.HydroError):
        B.hydro_gather(ok, 2, 7)
    empty = torch.zeros((5, 0, 16, 16), device="cuda")
    assert B.hydro_gather(empty, 2).shape[0] == 0


# the on-device driver against the host-gather loop of tests/harness.py (same kernels; dt/dh is formed on the device
# as cfl / max_speed instead of on the host as (cfl * dh / max_speed) / dh, so agreement is to rounding, not bitwise)
@pytest.mark.parametrize("dtype", (np.float32, np.float64))
def test_advance_matches_host_gather_loop(B, dtype):
    import torch
    gamma, N, steps = 5.0 / 3.0, 32, 6
    U0 = wl.blast_grid(N, dtype=dtype)
    Uh, th, _, _ = run_grid(CudaBackend(0), U0.copy(), steps, 1.0, gamma, CTU, HLLC, VANLEER, cfl=0.5)
    Ud, td = B.hydro_advance(torch.from_numpy(U0).cuda(), steps, 1.0, gamma, CTU, HLLC, VANLEER, cfl=0.5)
    d = np.abs(Ud.cpu().numpy().astype(np.float64) - Uh)
    tol = steps * (1e-5 if dtype == np.float32 else 1e-13)
    for v in ((0,), (1, 2, 3), (4,)):
        assert d[list(v)].sum() <= tol * np.abs(Uh[list(v)]).sum()
    assert abs(td.item() - th) <= 1e-6 * th


# config 1 on the device driver against the oracle (outflow ghosts, 20 steps, fp64)
def test_config1_sod_on_device(B):
    import torch
    from oracle import oracle as O
    gamma, N = 1.4, 32
    U0 = wl.sod_grid(N, axis=0, gamma=gamma)
    Ur, tr, _, _ = run_grid(OracleBackend(O, 4), U0.copy(), 20, 1.0 / N, gamma, CTU, ROE, VANLEER, cfl=0.5, bc="outflow")
    Ud, td = B.hydro_advance(torch.from_numpy(U0).cuda(), 20, 1.0 / N, gamma, CTU, ROE, VANLEER, cfl=0.5, bc=B.BC_OUTFLOW)
    d = np.abs(Ud.cpu().numpy() - Ur)
    for v, sc in ((0, np.abs(Ur[0]).max()), (1, np.abs(Ur[1:4]).max()), (4, np.abs(Ur[4]).max())):
        assert d[v].max() <= 20 * 1e-12 * sc
    assert abs(td.item() - tr) <= 1e-12 * tr


# config 2 at its FULL size (128^3 fp32, 50 steps, periodic) on the device: the properties that hold at any size
def test_config2_blast_full_size_properties(B):
    import torch
    gamma, N, steps = 5.0 / 3.0, 128, 50
    U0 = wl.blast_grid(N, dtype=np.float32)
    status = torch.zeros(3, dtype=torch.int64, device="cuda")
    Ud, _ = B.hydro_advance(torch.from_numpy(U0).cuda(), steps, 1.0, gamma, CTU, HLLC, VANLEER, cfl=0.5, status=status)
    U = Ud.cpu().numpy().astype(np.float64)
    assert status.cpu().tolist()[1] == 0 and np.isfinite(U).all() and U[0].min() > 0
    # conserved totals (P11): mass and energy drift, net momentum
    for v in (0, 4):
        s0 = U0[v].sum(dtype=np.float64)
        assert abs(U[v].sum() - s0) <= 1e-6 * s0
    assert np.abs(U[1:4].sum(axis=(1, 2, 3))).max() <= 1e-6 * np.abs(U[1:4]).sum()
    # axis-permutation and mirror symmetry (P14): rounding level in fp32, a direction bug gives O(1)
    rho = U[0]
    scale = np.abs(rho - 1.0).max()
    assert scale > 1e-2  # the blast has moved
    for perm in ((1, 0, 2), (2, 1, 0), (0, 2, 1), (1, 2, 0)):
        assert np.abs(rho - rho.transpose(perm)).max() <= 1e-4 * rho.max()
    # mirror about the grid node N/2 (the blast centre): cell i <-> N - 1 - i; the normal momentum changes sign
    assert np.abs(rho - rho[::-1, :, :]).max() <= 1e-4 * rho.max()
    assert np.abs(U[1] + U[1][:, :, ::-1]).max() <= 1e-4 * np.abs(U[1:4]).max()


def _totals(U):
    return [U[v].double().sum().item() for v in range(5)], U.abs().double().sum(dim=(1, 2, 3)).cpu().numpy()


# config 4 at its FULL size (256^3 fp32, periodic Kelvin-Helmholtz layer): every scheme x reconstruction x {Roe, HLLC},
# 10 steps each on the device; the properties that hold at any size (the element-wise parity of these variants is in
# test_gpu_parity.py: small KH box for 10 steps, and sampled groups of large batches)
@pytest.mark.parametrize("scheme", (0, 1, 2))
def test_config4_kh_full_size_properties(B, scheme):
    import torch
    gamma, N, steps = 1.4, 256, 10
    U0 = torch.from_numpy(wl.kh_grid((N, N, N), gamma=gamma, seed=1, dtype=np.float32)).cuda()
    tot0, abs0 = _totals(U0)
    for recon in (0, 1):
        for riemann in (ROE, HLLC):
            status = torch.zeros(3, dtype=torch.int64, device="cuda")
            # all 12 variants run in grid mode (one launch per step): the workspace is the second grid, no group buffers
            assert B.hydro_advance_workspace_bytes((N, N, N), torch.float32, scheme, VANLEER, recon=recon) == 256 + 5 * N ** 3 * 4
            U, t = B.hydro_advance(U0.clone(), steps, 1.0 / N, gamma, scheme, riemann, VANLEER, cfl=0.3, recon=recon,
                                   status=status)
            assert status.cpu().tolist()[1] == 0 and torch.isfinite(U).all().item()
            assert U[0].min().item() > 0.9 and t.item() > 0
            tot, _ = _totals(U)
            for v in (0, 1, 4):  # mass, x momentum, energy; y and z momenta start at ~0
                assert abs(tot[v] - tot0[v]) <= 2e-6 * abs0[v], (scheme, recon, riemann, v)
            for v in (2, 3):
                assert abs(tot[v] - tot0[v]) <= 2e-6 * abs0[1]
            # the shear layer is still there and the perturbation has not blown up
            assert 0.4 < U[1].abs().max().item() / U[0].max().item() < 0.7


# config 5 at its FULL size (512^3, 32768 patch groups, Mach-1 turbulence): CTU + PPM + exact solver, 10 steps, both precisions
@pytest.mark.parametrize("dtype", (np.float32, np.float64))
def test_config5_turbulence_full_size_properties(B, dtype):
    import torch
    gamma, N, steps = 5.0 / 3.0, 512, 10
    U0 = torch.from_numpy(wl.turbulence_grid(N, gamma=gamma, kmax=32, seed=2, dtype=dtype)).cuda()
    tot0, abs0 = _totals(U0)
    status = torch.zeros(3, dtype=torch.int64, device="cuda")
    U, t = B.hydro_advance(U0, steps, 1.0 / N, gamma, CTU, 0, VANLEER, cfl=0.5, recon=1, status=status)
    st = status.cpu().tolist()
    assert st[1] == 0 and st[2] == 0 and torch.isfinite(U).all().item() and U[0].min().item() > 0
    tot, _ = _totals(U)
    tol = 2e-6 if dtype == np.float32 else 1e-12
    for v in (0, 4):
        assert abs(tot[v] - tot0[v]) <= tol * abs0[v]
    for v in (1, 2, 3):
        assert abs(tot[v] - tot0[v]) <= tol * abs0[0]  # |v| ~ 1, rho = 1: the mass scale
    assert 0 < t.item() < 10 * 0.5 / N  # max speed >= c = 1


# CUDA-graph replay of the step (launch-bound small grids) gives the same bits as launching every step
def test_advance_graph_replay_is_identical(B):
    import torch
    gamma, N, steps = 1.4, 32, 12
    U0 = torch.from_numpy(wl.sod_grid(N, axis=1, gamma=gamma)).cuda()
    Ua, ta = B.hydro_advance(U0.clone(), steps, 1.0 / N, gamma, CTU, ROE, VANLEER, cfl=0.5, bc=B.BC_OUTFLOW)
    Ub, tb = B.hydro_advance(U0.clone(), steps, 1.0 / N, gamma, CTU, ROE, VANLEER, cfl=0.5, bc=B.BC_OUTFLOW, graph=True)
    assert torch.equal(Ua, Ub) and ta.item() == tb.item()


# hydro_solve_grid_* (ghost zones folded out of the grid inside the fused kernel, one launch) against the three-launch
# path gather -> hydro_solve -> scatter: same arithmetic on the same values, so the grids must agree bit for bit
@pytest.mark.parametrize("dtype", (np.float32, np.float64))
@pytest.mark.parametrize("bc", (0, 1))
@pytest.mark.parametrize("recon,riemann", ((0, ROE), (0, HLLC), (1, ROE), (1, 0)))
def test_solve_grid_equals_gather_solve_scatter(B, dtype, bc, recon, riemann):
    import torch
    gamma = 1.4
    U0 = torch.from_numpy(wl.kh_grid((32, 48, 64), gamma=gamma, seed=3, dtype=dtype)).cuda()  # Nz, Ny, Nx all different
    g = B.hydro_min_ghost(CTU, recon)
    groups = B.hydro_gather(U0, g, bc)
    smax = B.hydro_dt(groups, gamma, 0)
    dt = 0.4 * (1.0 / 64) / float(smax.item())
    st_a = torch.zeros(3, dtype=torch.int64, device="cuda")
    st_b = torch.zeros(3, dtype=torch.int64, device="cuda")
    na = torch.zeros((), dtype=U0.dtype, device="cuda")
    nb = torch.zeros((), dtype=U0.dtype, device="cuda")
    out, _ = B.hydro_solve(groups, dt, 1.0 / 64, gamma, CTU, riemann, VANLEER, recon=recon, face_flux=False, status=st_a,
                           next_max_speed=na)
    ref = B.hydro_scatter(out, tuple(U0.shape[1:]))
    got = B.hydro_solve_grid(U0, dt, 1.0 / 64, gamma, CTU, riemann, VANLEER, bc=bc, recon=recon, status=st_b, next_max_speed=nb)
    assert torch.equal(got, ref)
    assert st_a.tolist() == st_b.tolist() and na.item() == nb.item()


# round 2: every scheme and the non-default options (limiters, characteristic limiting, floors) in grid mode against
# gather -> hydro_solve -> scatter (the group path is what the parity tests compare with the oracle): bitwise for the default
# options, a few ulp for the others
@pytest.mark.parametrize("dtype", (np.float32, np.float64))
@pytest.mark.parametrize("scheme,recon,riemann,limiter,kw", (
    (0, 0, ROE, VANLEER, {}), (0, 1, HLLC, VANLEER, {}), (0, 0, ROE, 0, {}), (0, 1, ROE, 3, dict(char_limit=1)),
    (0, 0, HLLC, VANLEER, dict(min_dens=1e-3, min_pres=1e-3)),
    (1, 0, ROE, VANLEER, {}), (1, 1, HLLC, VANLEER, {}), (1, 0, ROE, 2, {}), (1, 1, ROE, 0, dict(char_limit=1)),
    (2, 0, ROE, 0, {}), (2, 1, HLLC, 2, dict(char_limit=1)), (2, 0, ROE, VANLEER, dict(min_dens=1e-3, min_pres=1e-3)),
    (2, 0, 1, 3, {})))
def test_solve_grid_all_schemes_and_options(B, dtype, scheme, recon, riemann, limiter, kw):
    import torch
    gamma = 1.4
    for bc in (0, 1):
        U0 = torch.from_numpy(wl.kh_grid((32, 48, 64), gamma=gamma, seed=5, dtype=dtype)).cuda()
        g = B.hydro_min_ghost(scheme, recon)
        groups = B.hydro_gather(U0, g, bc)
        smax = B.hydro_dt(groups, gamma, 1)
        dt = 0.8 * (1.0 / 64) / float(smax.item())
        st_a = torch.zeros(3, dtype=torch.int64, device="cuda")
        st_b = torch.zeros(3, dtype=torch.int64, device="cuda")
        na = torch.zeros((), dtype=U0.dtype, device="cuda")
        nb = torch.zeros((), dtype=U0.dtype, device="cuda")
        out, _ = B.hydro_solve(groups, dt, 1.0 / 64, gamma, scheme, riemann, limiter, recon=recon, face_flux=False, status=st_a,
                               next_max_speed=na, impl=B.IMPL_FUSED, **kw)
        ref = B.hydro_scatter(out, tuple(U0.shape[1:]))
        got = B.hydro_solve_grid(U0, dt, 1.0 / 64, gamma, scheme, riemann, limiter, bc=bc, recon=recon, status=st_b, next_max_speed=nb, **kw)
        if limiter == VANLEER and not kw:
            # default options: the kernels' own arithmetic (hydro_lean_math.cuh, explicit FMAs) is the same instruction sequence
            assert torch.equal(got, ref)
            assert na.item() == nb.item()
        else:
            # the other options run the generic arithmetic of hydro_math.cuh, written as plain a * b + c: the two template
            # instantiations may contract different multiply-add pairs into FMAs, so they agree to a few ulp, not bitwise
            eps = float(np.finfo(dtype).eps)
            assert (got.double() - ref.double()).abs().max().item() <= 8 * eps * ref.abs().max().item()
            assert abs(na.item() - nb.item()) <= 8 * eps * abs(na.item())
        assert st_a.tolist() == st_b.tolist()


def test_solve_grid_unsupported_variants(B):
    import torch
    U = torch.ones((5, 16, 16, 16), device="cuda")
    # the one variant without a grid mode: VL with positivity floors (its half step re-reads U^n of ghost cells from the batch)
    with pytest.raises(B.HydroError):
        B.hydro_solve_grid(U, 0.01, 1.0, 1.4, 1, ROE, VANLEER, min_dens=1e-3)
    with pytest.raises(B.HydroError):
        B.hydro_solve_grid(U, 0.01, 1.0, 1.4, CTU, ROE, VANLEER, out=U)
