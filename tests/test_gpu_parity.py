"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element, on the
same seeded inputs.  Tolerances are north_star's (BASELINE.json), in the readings S22 / S23 of DESIGN.md:
  fp64: per-variable max |gpu - ref| / max |ref| <= 1e-12 (the three momenta share one scale);
  fp32: per-variable L1  sum|gpu - ref| / sum|ref| <= 1e-5 per step against the fp32 oracle.
Integer results (status counters) are compared exactly.
"""
import itertools

import numpy as np
import pytest

from paper_1103_3373_b200 import workloads as wl
from tests.harness import CudaBackend, OracleBackend, run_grid

pytestmark = pytest.mark.gpu

MHM, VL, CTU = 0, 1, 2
EXACT, HLLE, HLLC, ROE = 0, 1, 2, 3
GMINMOD, VANLEER, VANALBADA, HYBRID = 0, 1, 2, 3
PLM, PPM = 0, 1
AUTO, STAGED, FUSED = 0, 1, 2
PS = 16
TOL64, TOL32 = 1e-12, 1e-5


@pytest.fixture(scope="module")
def B():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("gpu tests need a CUDA device")
    from paper_1103_3373_b200 import binding
    binding.lib()  # raises if the CUDA extension is missing: there is no fallback
    return binding


def err_max(a, b):
    """S22: per-variable max-norm relative error, momenta pooled.  a, b: [..., 5, *]-shaped with var axis 1."""
    d = np.abs(a.astype(np.float64) - b.astype(np.float64))
    sc = np.abs(b.astype(np.float64))
    ax = tuple(i for i in range(a.ndim) if i != 1)
    dm, sm = d.max(axis=ax), sc.max(axis=ax)
    scale = np.array([sm[0], sm[1:4].max(), sm[1:4].max(), sm[1:4].max(), sm[4]])
    return float((dm / scale).max())


def err_l1(a, b):
    """S23: per-variable L1 relative error, momenta pooled."""
    d = np.abs(a.astype(np.float64) - b.astype(np.float64))
    sc = np.abs(b.astype(np.float64))
    ax = tuple(i for i in range(a.ndim) if i != 1)
    ds, ss = d.sum(axis=ax), sc.sum(axis=ax)
    return float(max(ds[0] / ss[0], ds[1:4].sum() / ss[1:4].sum(), ds[4] / ss[4]))


def check(out, ff, ref_out, ref_ff, dtype, what):
    if dtype == np.float64:
        e = err_max(out, ref_out)
        assert e <= TOL64, (what, "out", e)
        # face_flux [Ng,9,5,16,16]: variable axis 2 -> move to 1
        e = err_max(np.moveaxis(ff, 2, 1), np.moveaxis(ref_ff, 2, 1))
        assert e <= TOL64, (what, "face_flux", e)
    else:
        e = err_l1(out, ref_out)
        assert e <= TOL32, (what, "out", e)
        e = err_l1(np.moveaxis(ff, 2, 1), np.moveaxis(ref_ff, 2, 1))
        assert e <= TOL32, (what, "face_flux", e)


def impls(B, dtype, scheme, recon, g=0):
    import torch
    t = {np.float32: torch.float32, np.float64: torch.float64}[dtype]
    r = (STAGED,)
    if B.hydro_fused_fits(t, scheme, recon, g):
        r += (FUSED,)
    return r


def gpu_solve(B, G, dt, dh, gamma, scheme, riemann, limiter, impl, **kw):
    return CudaBackend(impl).solve(G, dt, dh, gamma, scheme, riemann, limiter, **kw)


def amr(Ng, g, dtype, seed=0, gamma=5.0 / 3.0):
    return wl.amr_batch(Ng, g=g, gamma=gamma, seed=seed, dtype=np.dtype(dtype).name).numpy()


# ---- every variant, both precisions, small batch spanning several CTAs ---------------------------
@pytest.mark.parametrize("dtype", (np.float64, np.float32))
@pytest.mark.parametrize("scheme", (MHM, VL, CTU))
@pytest.mark.parametrize("recon", (PLM, PPM))
def test_all_variants_match_oracle(B, oracle, nthreads, dtype, scheme, recon):
    g = oracle.min_ghost(scheme, recon)
    gamma, dh = 5.0 / 3.0, 1.0
    G = amr(5, g, dtype, seed=11 + scheme)
    smax = oracle.hydro_dt(G, gamma, 0)
    dt = (0.5 if scheme == CTU else 0.3) * dh / smax
    for riemann, limiter, char in itertools.product((EXACT, HLLE, HLLC, ROE), (GMINMOD, VANLEER, VANALBADA, HYBRID), (0, 1)):
        ref_out, ref_ff, ref_st = oracle.hydro_solve(G, dt, dh, gamma, scheme, riemann, limiter, recon=recon,
                                                     char_limit=char, nthreads=nthreads)
        for impl in impls(B, dtype, scheme, recon):
            out, ff, st = gpu_solve(B, G, dt, dh, gamma, scheme, riemann, limiter, impl, recon=recon, char_limit=char)
            check(out, ff, ref_out, ref_ff, dtype, (scheme, recon, riemann, limiter, char, impl))
            assert st[1] == 0 and ref_st[1] == 0
            if impl == STAGED:  # same regions as the oracle -> identical event counts
                assert tuple(st[:3]) == tuple(ref_st[:3])


# ---- wider ghost zones than needed (config 3 supplies g = 3 to CTU+PLM), theta, fallbacks ---------
@pytest.mark.parametrize("dtype", (np.float64, np.float32))
def test_extra_ghosts_and_options(B, oracle, dtype):
    gamma, dh = 1.4, 0.5
    for scheme, recon, g in ((CTU, PLM, 3), (CTU, PLM, 4), (MHM, PPM, 4), (VL, PLM, 4)):
        G = amr(3, g, dtype, seed=5, gamma=gamma)
        dt = 0.3 * dh / oracle.hydro_dt(G, gamma, 0)
        for kw in (dict(minmod_coeff=1.0), dict(minmod_coeff=2.0), dict(roe_fallback=2), dict(roe_fallback=3)):
            ref = oracle.hydro_solve(G, dt, dh, gamma, scheme, ROE, GMINMOD, recon=recon, **kw)
            for impl in impls(B, dtype, scheme, recon, g):
                out, ff, st = gpu_solve(B, G, dt, dh, gamma, scheme, ROE, GMINMOD, impl, recon=recon, **kw)
                check(out, ff, ref[0], ref[1], dtype, (scheme, recon, g, kw, impl))


# ---- P1 on the GPU: uniform state is preserved bitwise by every variant -----------------------------
@pytest.mark.parametrize("dtype", (np.float64, np.float32))
def test_uniform_state_bitwise(B, dtype):
    gamma = 1.4
    for scheme, recon in itertools.product((MHM, VL, CTU), (PLM, PPM)):
        g = B.hydro_min_ghost(scheme, recon)
        S = PS + 2 * g
        one = np.ones((S, S, S), dtype)
        G = wl.prim_to_cons(1.3 * one, 0.4 * one, -0.7 * one, 0.2 * one, 0.9 * one, gamma)[None].astype(dtype)
        for riemann, impl in itertools.product((EXACT, HLLE, HLLC, ROE), impls(B, dtype, scheme, recon)):
            out, ff, st = gpu_solve(B, G, 0.01, 0.1, gamma, scheme, riemann, VANLEER, impl, recon=recon)
            assert np.array_equal(out, G[:, :, g:g + PS, g:g + PS, g:g + PS]), (scheme, recon, riemann, impl)
            assert not st.any()


# ---- edge cases: empty batch, one group, more groups than resident CTAs (ragged tail) ---------------
def test_batch_edges(B, oracle, nthreads):
    import torch
    gamma, dh = 5.0 / 3.0, 1.0
    empty = torch.empty((0, 5, 20, 20, 20), dtype=torch.float64, device="cuda")
    out, ff = B.hydro_solve(empty, 0.1, dh, gamma)
    assert out.shape == (0, 5, 16, 16, 16) and ff.shape == (0, 9, 5, 16, 16)
    assert B.hydro_dt(empty, gamma).item() == 0.0
    for Ng in (1, 2 * 148 * 4 + 37):
        G = amr(Ng, 2, np.float32, seed=3)
        dt = 0.4 * dh / oracle.hydro_dt(G, gamma, 0)
        ref = oracle.hydro_solve(G, dt, dh, gamma, CTU, HLLC, VANLEER, nthreads=nthreads)
        for impl in impls(B, np.float32, CTU, PLM):
            out, ff, st = gpu_solve(B, G, dt, dh, gamma, CTU, HLLC, VANLEER, impl)
            check(out, ff, ref[0], ref[1], np.float32, (Ng, impl))
            # every group individually (a wrong group offset would hide in a pooled norm)
            d = np.abs(out.astype(np.float64) - ref[0]).reshape(Ng, -1).max(1)
            assert d.max() <= 1e-4 * np.abs(ref[0]).max()
    # face_flux = NULL skips step (5) and leaves `out` unchanged
    G = amr(3, 2, np.float64, seed=4)
    a = gpu_solve(B, G, 0.05, dh, gamma, CTU, ROE, VANLEER, AUTO)
    b = gpu_solve(B, G, 0.05, dh, gamma, CTU, ROE, VANLEER, AUTO, want_flux=False)
    assert b[1] is None and np.array_equal(a[0], b[0])


# ---- A10: Roe failure -> fallback, counted identically (golden P8 data) ------------------
@pytest.mark.parametrize("fallback", (1, 2, 3))
def test_roe_failure_counts(B, oracle, fallback):
    gamma, g = 1.4, 2
    S = PS + 2 * g
    x = np.arange(S) - g
    vx = np.where(x < 8, -2.0, 2.0)[None, None, :] * np.ones((S, S, S))
    one = np.ones((S, S, S))
    G = wl.prim_to_cons(one, vx, 0 * one, 0 * one, 0.4 * one, gamma)[None]
    ref_out, ref_ff, ref_st = oracle.hydro_solve(G, 0.02, 1.0, gamma, CTU, ROE, VANLEER, roe_fallback=fallback)
    assert ref_st[0] > 0
    for impl in impls(B, np.float64, CTU, PLM):
        out, ff, st = gpu_solve(B, G, 0.02, 1.0, gamma, CTU, ROE, VANLEER, impl, roe_fallback=fallback)
        check(out, ff, ref_out, ref_ff, np.float64, ("roe-fail", fallback, impl))
        if impl == STAGED:
            assert tuple(st) == tuple(ref_st[:3])
        else:
            assert st[0] > 0


def test_floors_and_bad_state_counter(B, oracle):
    gamma, g = 1.4, 2
    G = amr(2, g, np.float64, seed=9, gamma=gamma)
    G[0, 4, 10, 10, 10] = 1e-9  # energy below kinetic -> negative pressure in one cell
    kw = dict(min_dens=1e-3, min_pres=1e-3)
    ref_out, ref_ff, ref_st = oracle.hydro_solve(G, 0.01, 1.0, gamma, CTU, HLLE, VANLEER, **kw)
    assert ref_st[1] > 0
    out, ff, st = gpu_solve(B, G, 0.01, 1.0, gamma, CTU, HLLE, VANLEER, STAGED, **kw)
    check(out, ff, ref_out, ref_ff, np.float64, "floors")
    assert st[1] == ref_st[1]


# ---- hydro_dt ----------------------------------------------------------------------------------------
@pytest.mark.parametrize("dtype", (np.float64, np.float32))
def test_hydro_dt(B, oracle, dtype):
    import torch
    gamma = 5.0 / 3.0
    for Ng, g in ((1, 0), (7, 2), (300, 3)):
        G = amr(Ng, g, dtype, seed=21)
        t = torch.from_numpy(G).cuda()
        for norm in (0, 1):
            got = B.hydro_dt(t, gamma, norm).item()
            ref = oracle.hydro_dt(G, gamma, norm)
            assert abs(got - ref) <= 4 * np.finfo(dtype).eps * ref, (Ng, g, norm, got, ref)
    # ghost cells are not scanned; a bad interior cell gives NaN
    G = amr(4, 2, dtype, seed=22)
    G2 = G.copy()
    G2[:, 1, 0, 0, 0] = 1e6
    assert B.hydro_dt(torch.from_numpy(G2).cuda(), gamma).item() == B.hydro_dt(torch.from_numpy(G).cuda(), gamma).item()
    G2 = G.copy()
    G2[3, 0, 5, 5, 5] = -1.0
    assert np.isnan(B.hydro_dt(torch.from_numpy(G2).cuda(), gamma).item())


# ---- config 1: Sod on 32^3 fp64, CTU+PLM(van Leer)+Roe, CFL 0.5, 20 steps, every step ----------------
@pytest.mark.parametrize("axis", (0, 1, 2))
def test_config1_sod_every_step(B, oracle, nthreads, axis):
    gamma, N = 1.4, 32
    U0 = wl.sod_grid(N, axis=axis, gamma=gamma, dtype=np.float64)
    ref_steps = []
    run_grid(OracleBackend(oracle, nthreads), U0.copy(), 20, 1.0 / N, gamma, CTU, ROE, VANLEER, cfl=0.5, bc="outflow",
             on_step=lambda s, U, ff, G, dt: ref_steps.append((U.copy(), ff.copy(), dt)))
    for impl in impls(B, np.float64, CTU, PLM):
        def cmp(s, U, ff, G, dt):
            Ur, ffr, dtr = ref_steps[s]
            assert abs(dt - dtr) <= 1e-14 * dtr
            assert err_max(U[None], Ur[None]) <= TOL64, (axis, impl, s)
            assert err_max(np.moveaxis(ff, 2, 1), np.moveaxis(ffr, 2, 1)) <= TOL64, (axis, impl, s)
        run_grid(CudaBackend(impl), U0.copy(), 20, 1.0 / N, gamma, CTU, ROE, VANLEER, cfl=0.5, bc="outflow", on_step=cmp)


# ---- config 2 shape at reduced size: blast, fp32, CTU+PLM+HLLC, periodic, multi-step -------------------
def test_config2_blast_small(B, oracle, nthreads):
    gamma, N, steps = 5.0 / 3.0, 32, 12
    U0 = wl.blast_grid(N, radius=3.0, gamma=gamma, dtype=np.float32)
    Ur, _, str_, _ = run_grid(OracleBackend(oracle, nthreads), U0.copy(), steps, 1.0, gamma, CTU, HLLC, VANLEER, cfl=0.5)
    for impl in impls(B, np.float32, CTU, PLM):
        Ug, _, stg, _ = run_grid(CudaBackend(impl), U0.copy(), steps, 1.0, gamma, CTU, HLLC, VANLEER, cfl=0.5)
        assert err_l1(Ug[None], Ur[None]) <= steps * TOL32, impl
        assert stg[1] == 0
        # P11 on the GPU result: conserved totals (fp64 accumulation)
        for v in (0, 4):
            assert abs(Ug[v].sum(dtype=np.float64) - U0[v].sum(dtype=np.float64)) <= 1e-6 * U0[v].sum(dtype=np.float64)


# ---- config 4 shape at reduced size: KH box, all 12 scheme x recon x solver variants, 10 steps --------
@pytest.mark.parametrize("scheme", (MHM, VL, CTU))
@pytest.mark.parametrize("recon", (PLM, PPM))
def test_config4_kh_small(B, oracle, nthreads, scheme, recon):
    gamma, steps = 1.4, 10
    U0 = wl.kh_grid((16, 64, 32), gamma=gamma, seed=1, dtype=np.float32)
    dh = 1.0 / 256
    for riemann in (ROE, HLLC):
        Ur, _, _, _ = run_grid(OracleBackend(oracle, nthreads), U0.copy(), steps, dh, gamma, scheme, riemann, VANLEER,
                               recon=recon, cfl=0.3)
        for impl in impls(B, np.float32, scheme, recon):
            Ug, _, st, _ = run_grid(CudaBackend(impl), U0.copy(), steps, dh, gamma, scheme, riemann, VANLEER,
                                    recon=recon, cfl=0.3)
            assert err_l1(Ug[None], Ur[None]) <= steps * TOL32, (scheme, recon, riemann, impl)


# ---- config 5 shape at reduced size: turbulence 32^3, CTU+PPM+exact with hydro_dt, both precisions ----
@pytest.mark.parametrize("dtype", (np.float64, np.float32))
def test_config5_turbulence_small(B, oracle, nthreads, dtype):
    gamma, N, steps = 5.0 / 3.0, 32, 5
    U0 = wl.turbulence_grid(N, gamma=gamma, kmax=8, seed=2, dtype=dtype)
    Ur, _, str_, _ = run_grid(OracleBackend(oracle, nthreads), U0.copy(), steps, 1.0 / N, gamma, CTU, EXACT, VANLEER,
                              recon=PPM, cfl=0.5)
    for impl in impls(B, dtype, CTU, PPM):
        Ug, _, stg, _ = run_grid(CudaBackend(impl), U0.copy(), steps, 1.0 / N, gamma, CTU, EXACT, VANLEER, recon=PPM,
                                 cfl=0.5)
        if dtype == np.float64:
            assert err_max(Ug[None], Ur[None]) <= TOL64, impl  # the bar itself after 5 steps, as config 1 after 20
        else:
            assert err_l1(Ug[None], Ur[None]) <= steps * TOL32, impl
        assert stg[2] == 0 and str_[2] == 0


# ---- the host-buffer pipeline gives the device path's bits -------------------------------------------
@pytest.mark.parametrize("dtype", (np.float64, np.float32))
def test_pipeline_matches_device_path(B, dtype):
    import torch
    gamma, g, Ng = 5.0 / 3.0, 3, 37
    Gt = wl.amr_batch(Ng, g=g, gamma=gamma, seed=8, dtype=np.dtype(dtype).name)
    dev_out, dev_ff = B.hydro_solve(Gt.cuda(), 0.1, 1.0, gamma, CTU, ROE, VANLEER)
    pipe = B.HydroPipeline(Gt.dtype, g, groups_per_chunk=8, nstreams=3)
    hin = Gt.pin_memory()
    hout = torch.empty((Ng, 5, PS, PS, PS), dtype=Gt.dtype).pin_memory()
    hff = torch.empty((Ng, 9, 5, PS, PS), dtype=Gt.dtype).pin_memory()
    st = torch.zeros(3, dtype=torch.int64)
    pipe.solve(hin, hout, hff, 0.1, 1.0, gamma, CTU, ROE, VANLEER, status=st)
    assert torch.equal(hout, dev_out.cpu()) and torch.equal(hff, dev_ff.cpu())
    pipe.close()


# ---- config 3 at BASELINE.json's full size, in the launch configuration bench.py times ---------------
# 8192 groups, g = 3, hydro_dt -> hydro_solve with dt formed on the device (max_speed + cfl), AUTO kernel choice,
# face fluxes on.  Groups are independent, so sampled groups are compared element by element with the oracle; the
# conservation balance that ties `out` to `face_flux` (P11) is checked on ALL groups.
@pytest.mark.parametrize("dtype", (np.float32, np.float64))
def test_config3_full_size_sampled(B, oracle, nthreads, dtype):
    import torch
    Ng, g, gamma, dh, cfl = 8192, 3, 5.0 / 3.0, 1.0, 0.5
    tdt = torch.float32 if dtype == np.float32 else torch.float64
    u = wl.amr_batch(Ng, g=g, gamma=gamma, seed=0, dtype=np.dtype(dtype).name, device=torch.device("cuda"))
    smax = torch.empty((), dtype=tdt, device="cuda")
    status = torch.zeros(3, dtype=torch.int64, device="cuda")
    B.hydro_dt(u, gamma, 0, max_speed=smax)
    out, ff = B.hydro_solve(u, 0.0, dh, gamma, CTU, ROE, VANLEER, status=status, max_speed=smax, cfl=cfl)
    torch.cuda.synchronize()
    assert status.cpu().tolist() == [0, 0, 0]
    # the whole-batch reduction against the oracle's (order-independent maximum)
    rng = np.random.default_rng(7)
    pick = np.sort(np.unique(np.concatenate([[0, 1, 147, 148, 295, 296, Ng - 1], rng.choice(Ng, 60, replace=False)])))[:64]  # 64 groups
    Gs = u[torch.from_numpy(pick).cuda()].cpu().numpy()
    s_gpu = dtype(smax.item())
    s_ref = max(oracle.hydro_dt(u[k:k + 512].cpu().numpy(), gamma, 0) for k in range(0, Ng, 512))
    assert abs(float(s_gpu) - s_ref) <= 4 * np.finfo(dtype).eps * s_ref
    dt = float(dtype(cfl) / s_gpu)  # the kernel forms nu = cfl / max_speed in the working precision; dh = 1
    ref_out, ref_ff, ref_st = oracle.hydro_solve(Gs, dt, dh, gamma, CTU, ROE, VANLEER, nthreads=nthreads)[:3]
    idx = torch.from_numpy(pick).cuda()
    check(out[idx].cpu().numpy(), ff[idx].cpu().numpy(), ref_out, ref_ff, dtype, ("config3 full size", np.dtype(dtype).name))
    d = np.abs(out[idx].cpu().numpy().astype(np.float64) - ref_out).reshape(len(pick), -1).max(1)
    assert d.max() <= (1e-4 if dtype == np.float32 else 1e-11) * np.abs(ref_out).max()
    # P11 on every group: sum_interior(out - in) = -nu * (signed sum of the six outer flux planes)
    o64, f64 = out.double(), ff.double()
    uin = u[:, :, g:g + PS, g:g + PS, g:g + PS].double()
    lhs = (o64 - uin).sum(dim=(2, 3, 4))
    net = sum(f64[:, 3 * d + 2].sum(dim=(2, 3)) - f64[:, 3 * d + 0].sum(dim=(2, 3)) for d in range(3))
    nu = float(dtype(cfl) / s_gpu) / dh
    scale = uin.abs().sum(dim=(2, 3, 4)).max().item()
    tol = (2e-6 if dtype == np.float32 else 1e-13) * scale
    assert (lhs + nu * net).abs().max().item() <= tol


# ---- the other schemes / reconstructions / solvers on a batch that fills the persistent grid many times over -------
# (the kernels of configs 4 and 5: MHM, VL, PPM, HLLC, exact), sampled groups against the oracle, flux balance on all.
@pytest.mark.parametrize("dtype", (np.float32, np.float64))
@pytest.mark.parametrize("scheme,recon,riemann", ((MHM, PLM, HLLC), (MHM, PPM, ROE), (VL, PLM, ROE), (VL, PPM, HLLC),
                                                  (CTU, PPM, EXACT), (CTU, PPM, ROE)))
def test_large_batch_sampled_variants(B, oracle, nthreads, dtype, scheme, recon, riemann):
    import torch
    Ng, gamma, dh = 2048, 5.0 / 3.0, 1.0
    g = oracle.min_ghost(scheme, recon)
    tdt = torch.float32 if dtype == np.float32 else torch.float64
    assert B.hydro_fused_fits(tdt, scheme, recon, g)
    u = wl.amr_batch(Ng, g=g, gamma=gamma, seed=5, dtype=np.dtype(dtype).name, device=torch.device("cuda"))
    status = torch.zeros(3, dtype=torch.int64, device="cuda")
    dt = 0.3 * dh / float(B.hydro_dt(u, gamma, 0).item())  # CFL 0.3: stable for MHM and VL too (S15)
    out, ff = B.hydro_solve(u, dt, dh, gamma, scheme, riemann, VANLEER, recon=recon, status=status, impl=FUSED)
    torch.cuda.synchronize()
    st = status.cpu().tolist()
    assert st[1] == 0 and st[2] == 0
    pick = np.sort(np.concatenate([[0, 147, 148, 296, Ng - 1], np.random.default_rng(11).choice(Ng, 11, replace=False)]))
    idx = torch.from_numpy(pick).cuda()
    ref_out, ref_ff, _ = oracle.hydro_solve(u[idx].cpu().numpy(), dt, dh, gamma, scheme, riemann, VANLEER, recon=recon,
                                            nthreads=nthreads)[:3]
    check(out[idx].cpu().numpy(), ff[idx].cpu().numpy(), ref_out, ref_ff, dtype, (scheme, recon, riemann, np.dtype(dtype).name))
    uin = u[:, :, g:g + PS, g:g + PS, g:g + PS].double()
    lhs = (out.double() - uin).sum(dim=(2, 3, 4))
    f64 = ff.double()
    net = sum(f64[:, 3 * d + 2].sum(dim=(2, 3)) - f64[:, 3 * d + 0].sum(dim=(2, 3)) for d in range(3))
    scale = uin.abs().sum(dim=(2, 3, 4)).max().item()
    assert (lhs + (dt / dh) * net).abs().max().item() <= (2e-6 if dtype == np.float32 else 1e-13) * scale


# ---- hydro_opts::next_max_speed: the update's fused wave-speed reduction equals hydro_dt of `out` ----------------
@pytest.mark.parametrize("dtype", (np.float32, np.float64))
@pytest.mark.parametrize("scheme", (MHM, VL, CTU))
def test_next_max_speed_matches_hydro_dt(B, dtype, scheme):
    import torch
    gamma, dh = 5.0 / 3.0, 1.0
    tdt = torch.float32 if dtype == np.float32 else torch.float64
    g = B.hydro_min_ghost(scheme, PLM)
    u = wl.amr_batch(301, g=g, gamma=gamma, seed=9, dtype=np.dtype(dtype).name, device=torch.device("cuda"))
    dt = 0.3 * dh / float(B.hydro_dt(u, gamma, 0).item())
    for impl in impls(B, dtype, scheme, PLM):
        for norm in (0, 1):
            nxt = torch.full((), -1.0, dtype=tdt, device="cuda")
            out, _ = B.hydro_solve(u, dt, dh, gamma, scheme, ROE, VANLEER, impl=impl, face_flux=False,
                                   next_max_speed=nxt, next_norm=norm)
            ref = B.hydro_dt(out, gamma, norm).item()
            assert abs(nxt.item() - ref) <= 16 * np.finfo(dtype).eps * ref, (scheme, impl, norm)
    # a bad updated cell must surface as NaN, as in hydro_dt
    bad = u.clone()
    bad[7, 4] = -1.0  # negative energy everywhere in one group -> negative pressure after the update
    nxt = torch.zeros((), dtype=tdt, device="cuda")
    B.hydro_solve(bad, dt, dh, gamma, scheme, HLLE, VANLEER, face_flux=False, next_max_speed=nxt)
    assert np.isnan(nxt.item())
