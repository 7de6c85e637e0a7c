"""Pins for the directionally split relaxing-TVD oracle (oracle/rtvd_oracle.cpp).

The paper names the scheme (Jin & Xin 1995) and gives no formulas; the oracle follows reading S26 of DESIGN.md.  What pins it:
the uniform-state identity, exact conservation (update tied to the stored fluxes), mirror symmetry (right and left movers
treated alike), second-order convergence on a smooth wave (the limiter corrections and the midpoint rule: a first-order
flux or a full-step predictor drops the rate to ~1) and the Sod solution against the exact Riemann solution (the flux
function and the freezing speed: a wrong pressure term or wave speed moves the shock).
"""
import numpy as np
import pytest

from paper_1103_3373_b200 import workloads as wl
from tests.harness import run_grid


class RtvdBackend:
    """hydro_dt + split RTVD step behind the two calls run_grid makes; sweep order alternates x,y,z / z,y,x per step."""

    def __init__(self, O, nthreads=1, alternate=True):
        self.O, self.nthreads, self.alternate, self.step = O, nthreads, alternate, 0

    def dt(self, G, gamma, norm):
        return self.O.hydro_dt(G, gamma, norm)

    def solve(self, G, dt, dh, gamma, scheme, riemann, limiter, **kw):
        order = (self.step & 1) if self.alternate else 0
        self.step += 1
        return self.O.rtvd_solve(G, dt, dh, gamma, order=order, nthreads=self.nthreads)


def test_uniform_state_is_preserved_bitwise(oracle):
    G = np.empty((2, 5, 22, 22, 22))
    for q, v in enumerate((1.3, 0.4, -0.7, 0.2, 2.9)):
        G[:, q] = v
    for order in (0, 1):
        out, ff, st = oracle.rtvd_solve(G, 0.05, 1.0, 1.4, order=order)
        assert np.array_equal(out, G[:, :, 3:19, 3:19, 3:19]) and st[1] == 0
        # the stored flux of a uniform state is its physical flux
        rho, v, E = 1.3, np.array([0.4, -0.7, 0.2]) / 1.3, 2.9
        P = 0.4 * (E - 0.5 * rho * (v ** 2).sum())
        for d in range(3):
            assert np.allclose(ff[:, 3 * d:3 * d + 3, 0], rho * v[d], rtol=1e-14)
            assert np.allclose(ff[:, 3 * d:3 * d + 3, 1 + d], rho * v[d] ** 2 + P, rtol=1e-14)
            assert np.allclose(ff[:, 3 * d:3 * d + 3, 4], (E + P) * v[d], rtol=1e-14)


@pytest.mark.parametrize("order", (0, 1))
def test_update_equals_the_stored_flux_balance(oracle, order):
    gamma = 5.0 / 3.0
    G = wl.amr_batch(4, g=3, gamma=gamma, seed=17, dtype="float64").numpy()
    dt = 0.3 / oracle.hydro_dt(G, gamma, 0)
    out, ff, st = oracle.rtvd_solve(G, dt, 1.0, gamma, order=order)
    lhs = (out - G[:, :, 3:19, 3:19, 3:19]).sum(axis=(2, 3, 4))
    net = sum(ff[:, 3 * d + 2].sum(axis=(2, 3)) - ff[:, 3 * d].sum(axis=(2, 3)) for d in range(3))
    assert np.abs(lhs + dt * net).max() <= 1e-13 * np.abs(G).sum(axis=(2, 3, 4)).max()
    assert st[1] == 0


def test_periodic_conservation_and_mirror_symmetry(oracle, nthreads):
    gamma, N = 1.4, 32
    U0 = wl.kh_grid((N, N, N), gamma=gamma, seed=4, dtype=np.float64)
    U0[0] += 0.2 * np.sin(2 * np.pi * (np.arange(N) + 0.5) / N)[None, None, :]  # break the symmetry along x
    U, t, st, _ = run_grid(RtvdBackend(oracle, nthreads), U0.copy(), 6, 1.0 / N, gamma, 3, 0, 0, cfl=0.3, g=3)
    for v in range(5):
        assert abs(U[v].sum() - U0[v].sum()) <= 1e-13 * np.abs(U0[v]).sum() + 1e-13 * np.abs(U0[1]).sum()
    # mirror the data in x (cell i <-> N-1-i, x momentum negated): the result is the mirror image, to rounding
    M0 = U0[:, :, :, ::-1].copy()
    M0[1] *= -1
    M, _, _, _ = run_grid(RtvdBackend(oracle, nthreads), M0, 6, 1.0 / N, gamma, 3, 0, 0, cfl=0.3, g=3)
    back = M[:, :, :, ::-1].copy()
    back[1] *= -1
    assert np.abs(back - U).max() <= 1e-12 * np.abs(U).max()


def test_second_order_convergence(oracle, nthreads):
    # entropy wave carried diagonally through a periodic unit box for one period; sweep orders alternate (Strang)
    gamma, A = 5.0 / 3.0, 0.1
    v = np.array([1.0, 1.0, 1.0])      # diagonal advection, period 1
    errs = []
    for N in (16, 32):
        x = (np.arange(N) + 0.5) / N
        Z, Y, X = np.meshgrid(x, x, x, indexing="ij")
        rho = 1.0 + A * np.sin(2 * np.pi * (X + Y + Z))
        one = np.ones_like(rho)
        U0 = wl.prim_to_cons(rho, v[0] * one, v[1] * one, v[2] * one, 0.6 * one, gamma)
        dh = 1.0 / N
        smax = 1.0 + np.sqrt(gamma * 0.6 / (1 - A))
        nsteps = int(np.ceil(1.0 / (0.4 * dh / smax) / 2) * 2)  # even: complete x,y,z / z,y,x pairs
        U, t, _, _ = run_grid(RtvdBackend(oracle, nthreads), U0.copy(), nsteps, dh, gamma, 3, 0, 0, g=3, fixed_dt=1.0 / nsteps)
        errs.append(np.abs(U[0] - U0[0]).mean())
    rate = np.log2(errs[0] / errs[1])
    print("rtvd convergence", errs, rate)
    assert rate > 1.6, (errs, rate)   # van Leer clips the extrema: slightly below 2 in L1
    assert errs[1] < 0.1 * A          # the relaxing scheme is diffusive (c = |v| + cs), but the wave survives a period


def test_sod_against_the_exact_solution(oracle, nthreads):
    gamma = 1.4
    errs = []
    for N in (32, 64):
        U0 = wl.sod_grid(N, axis=0, gamma=gamma)[:, :16, :16, :] if N > 16 else wl.sod_grid(N, axis=0, gamma=gamma)
        U0 = np.ascontiguousarray(U0)
        U, t, st, _ = run_grid(RtvdBackend(oracle, nthreads), U0.copy(), int(0.6 * N), 1.0 / N, gamma, 3, 0, 0, cfl=0.4,
                               bc="outflow", g=3)
        assert st[1] == 0
        x = (np.arange(N) + 0.5) / N
        # exact solution sampled cell by cell with the oracle's exact Riemann sampler on the self-similar variable
        WL, WR = np.array([1.0, 0, 0, 0, 1.0]), np.array([0.125, 0, 0, 0, 0.1])
        rho_ex = np.array([sample(oracle, WL, WR, gamma, (xi - 0.5) / t) for xi in x])
        errs.append(np.abs(U[0, 0, 0, :] - rho_ex).mean())
        assert np.abs(U[0] - U[0, :1, :1, :]).max() <= 1e-13  # stays one-dimensional
    assert errs[0] < 2.5e-2 and errs[1] < 0.7 * errs[0], errs


def sample(oracle, WL, WR, gamma, xi):
    """Density of the exact solution at x/t = xi: shift to the frame moving with xi, sample at x/t = 0."""
    a, b = WL.copy(), WR.copy()
    a[1] -= xi
    b[1] -= xi
    rc, W = oracle.exact_sample0(a, b, gamma)
    return W[0]
