"""Pins for the directionally split weighted-average-flux oracle (oracle/waf_oracle.cpp).

The paper names the scheme (Toro 2009) and gives no formulas; the oracle follows reading S29 of DESIGN.md.  What pins it: the
uniform-state identity; exact conservation (update tied to the stored fluxes); mirror symmetry (waves 1 and 3, upwind choice);
a moving contact against the flux-limited Lax-Wendroff closed form written here in NumPy (the HLLC solution of a contact is
exact, so WAF must reduce to the scalar scheme: this fixes the limiter, the upwind ratio, the Courant weights and the
tangential-momentum rule); second-order convergence on a smooth wave (A = 1 everywhere is the first-order Godunov flux: rate ~1) and the
Sod solution against the exact Riemann solution (wave speeds and star states)."""
import numpy as np
import pytest

from paper_1103_3373_b200 import workloads as wl
from tests.harness import run_grid
from tests.test_oracle_rtvd import sample


class WafBackend:
    """hydro_dt + split WAF step behind the two calls run_grid makes; sweep order alternates x,y,z / z,y,x per step."""

    def __init__(self, O, nthreads=1, alternate=True):
        self.O, self.nthreads, self.alternate, self.step = O, nthreads, alternate, 0

    def dt(self, G, gamma, norm):
        return self.O.hydro_dt(G, gamma, norm)

    def solve(self, G, dt, dh, gamma, scheme, riemann, limiter, **kw):
        order = (self.step & 1) if self.alternate else 0
        self.step += 1
        return self.O.waf_solve(G, dt, dh, gamma, order=order, nthreads=self.nthreads)


def test_uniform_state_is_preserved_bitwise(oracle):
    G = np.empty((2, 5, 22, 22, 22))
    for q, v in enumerate((1.3, 0.4, -0.7, 0.2, 2.9)):
        G[:, q] = v
    for order in (0, 1):
        out, ff, st = oracle.waf_solve(G, 0.05, 1.0, 1.4, order=order)
        assert np.array_equal(out, G[:, :, 3:19, 3:19, 3:19]) and st[1] == 0
        rho, v, E = 1.3, np.array([0.4, -0.7, 0.2]) / 1.3, 2.9
        P = 0.4 * (E - 0.5 * rho * (v ** 2).sum())
        for d in range(3):  # the stored flux of a uniform state is its physical flux
            assert np.allclose(ff[:, 3 * d:3 * d + 3, 0], rho * v[d], rtol=1e-14)
            assert np.allclose(ff[:, 3 * d:3 * d + 3, 1 + d], rho * v[d] ** 2 + P, rtol=1e-14)
            assert np.allclose(ff[:, 3 * d:3 * d + 3, 4], (E + P) * v[d], rtol=1e-14)


@pytest.mark.parametrize("order", (0, 1))
def test_update_equals_the_stored_flux_balance(oracle, order):
    gamma = 5.0 / 3.0
    G = wl.amr_batch(4, g=3, gamma=gamma, seed=17, dtype="float64").numpy()
    dt = 0.3 / oracle.hydro_dt(G, gamma, 0)
    out, ff, st = oracle.waf_solve(G, dt, 1.0, gamma, order=order)
    lhs = (out - G[:, :, 3:19, 3:19, 3:19]).sum(axis=(2, 3, 4))
    net = sum(ff[:, 3 * d + 2].sum(axis=(2, 3)) - ff[:, 3 * d].sum(axis=(2, 3)) for d in range(3))
    assert np.abs(lhs + dt * net).max() <= 1e-13 * np.abs(G).sum(axis=(2, 3, 4)).max()
    assert st[1] == 0


def test_periodic_conservation_and_mirror_symmetry(oracle, nthreads):
    gamma, N = 1.4, 32
    U0 = wl.kh_grid((N, N, N), gamma=gamma, seed=4, dtype=np.float64)
    U0[0] += 0.2 * np.sin(2 * np.pi * (np.arange(N) + 0.5) / N)[None, None, :]  # break the symmetry along x
    U, t, st, _ = run_grid(WafBackend(oracle, nthreads), U0.copy(), 6, 1.0 / N, gamma, 3, 0, 0, cfl=0.3, g=3)
    for v in range(5):
        assert abs(U[v].sum() - U0[v].sum()) <= 1e-13 * np.abs(U0[v]).sum() + 1e-13 * np.abs(U0[1]).sum()
    M0 = U0[:, :, :, ::-1].copy()   # mirror in x (cell i <-> N-1-i, x momentum negated): the result is the mirror image
    M0[1] *= -1
    M, _, _, _ = run_grid(WafBackend(oracle, nthreads), M0, 6, 1.0 / N, gamma, 3, 0, 0, cfl=0.3, g=3)
    back = M[:, :, :, ::-1].copy()
    back[1] *= -1
    assert np.abs(back - U).max() <= 1e-12 * np.abs(U).max()


def _limited_lw(q, c):
    """One step of the flux-limited Lax-Wendroff scheme for q_t + u q_x = 0 on a pencil, Courant number c = u dt/dx of either
    sign, van Leer limiter B(r) = 2r/(1+r) (r > 0), written from the textbook: the face value between cells L = f-1 and R = f is
    q_L + (1 - |c|) B(r)/2 (q_R - q_L) for c > 0 and q_R - (1 - |c|) B(r)/2 (q_R - q_L) for c < 0, r = upwind jump / local jump.
    Returns the face values for f = 2 .. n-2 (index f)."""
    n = len(q)
    face = np.zeros(n)
    for f in range(2, n - 1):
        b = q[f] - q[f - 1]
        a = (q[f - 1] - q[f - 2]) if c > 0 else (q[f + 1] - q[f])
        B = 2 * a / (a + b) if a * b > 0 else 0.0
        face[f] = q[f - 1] + 0.5 * (1 - abs(c)) * B * b if c > 0 else q[f] - 0.5 * (1 - abs(c)) * B * b
    return face


@pytest.mark.parametrize("d", (0, 1, 2))
@pytest.mark.parametrize("sign", (1.0, -1.0))
def test_moving_contact_reduces_to_limited_lax_wendroff(oracle, d, sign):
    # uniform pressure and normal velocity u; density AND the two tangential velocities vary along the sweep direction d:
    # the HLLC solution of every face is the exact contact, so one sweep must advect rho, rho v_t1, rho v_t2 with the scalar
    # scheme above, each limited on its own jumps (S29)
    gamma, P, u, nu = 1.4, 1.0, 0.7 * sign, 0.4
    rng = np.random.default_rng(5)
    n = 22
    rho = 1.0 + 0.5 * rng.random(n)
    v1 = 0.3 * rng.standard_normal(n)
    v2 = 0.3 * rng.standard_normal(n)
    t1, t2 = (1 if d == 0 else 0), (1 if d == 2 else 2)
    shape = [1, 1, 1]
    shape[2 - d] = n   # array axes are (z, y, x)
    G = np.empty((1, 5, n, n, n))
    vel = [None, None, None]
    vel[d], vel[t1], vel[t2] = u * np.ones(n), v1, v2
    G[0, 0] = rho.reshape(shape)
    for a in range(3):
        G[0, 1 + a] = (rho * vel[a]).reshape(shape)
    G[0, 4] = (P / (gamma - 1) + 0.5 * rho * (u * u + v1 * v1 + v2 * v2)).reshape(shape)
    # sweeping d FIRST: order 0 for d = x, order 1 for d = z; for d = y compare the stored y flux of a state uniform in x and z
    # (the x sweep before it and the z sweep after it leave such a state untouched in the interior)
    order = 1 if d == 2 else 0
    out, ff, st = oracle.waf_solve(G, nu, 1.0, gamma, order=order)
    c = nu * u
    # every transported quantity is limited on its OWN jumps: rho on the density jumps, rho v_t on the jumps of rho v_t (S29)
    fr, f1, f2 = _limited_lw(rho, c), _limited_lw(rho * v1, c), _limited_lw(rho * v2, c)
    for s, f in enumerate((3, 11, 19)):   # stored planes: faces 0, 8, 16 of the interior = pencil faces 3, 11, 19
        got = ff[0, 3 * d + s]
        assert np.allclose(got[0], u * fr[f], rtol=1e-13, atol=1e-14)
        assert np.allclose(got[1 + t1], u * f1[f], rtol=1e-12, atol=1e-13)
        assert np.allclose(got[1 + t2], u * f2[f], rtol=1e-12, atol=1e-13)
        assert np.allclose(got[1 + d], u * u * fr[f] + P, rtol=1e-13)
    # and the density update of the interior cells of the pencil
    new = rho.copy()
    new[3:19] = rho[3:19] - c * (fr[4:20] - fr[3:19])
    sl = [slice(3, 19)] * 3
    got_rho = out[0, 0]
    ref = new[3:19].reshape([16 if k == 2 - d else 1 for k in range(3)])
    assert np.allclose(got_rho, np.broadcast_to(ref, got_rho.shape), rtol=1e-13)


def test_second_order_convergence(oracle, nthreads):
    gamma, A = 5.0 / 3.0, 0.1
    v = np.array([1.0, 1.0, 1.0])      # diagonal advection of an entropy wave, period 1
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
        U, t, _, _ = run_grid(WafBackend(oracle, nthreads), U0.copy(), nsteps, dh, gamma, 3, 0, 0, g=3, fixed_dt=1.0 / nsteps)
        errs.append(np.abs(U[0] - U0[0]).mean())
    rate = np.log2(errs[0] / errs[1])
    print("waf convergence", errs, rate)
    # the van Leer limiter clips the extrema of the wave, which holds the L1 rate below 2 at these resolutions (observed 1.58);
    # the first-order scheme (A = 1 everywhere) has a rate below 1 and an error of the order of the amplitude itself
    assert rate > 1.4, (errs, rate)
    assert errs[1] < 0.07 * A


def test_sod_against_the_exact_solution(oracle, nthreads):
    gamma = 1.4
    errs = []
    for N in (32, 64):
        U0 = np.ascontiguousarray(wl.sod_grid(N, axis=0, gamma=gamma)[:, :16, :16, :])
        U, t, st, _ = run_grid(WafBackend(oracle, nthreads), U0.copy(), int(0.6 * N), 1.0 / N, gamma, 3, 0, 0, cfl=0.4,
                               bc="outflow", g=3)
        assert st[1] == 0
        x = (np.arange(N) + 0.5) / N
        WL, WR = np.array([1.0, 0, 0, 0, 1.0]), np.array([0.125, 0, 0, 0, 0.1])
        rho_ex = np.array([sample(oracle, WL, WR, gamma, (xi - 0.5) / t) for xi in x])
        errs.append(np.abs(U[0, 0, 0, :] - rho_ex).mean())
        assert np.abs(U[0] - U[0, :1, :1, :]).max() <= 1e-13  # stays one-dimensional
    assert errs[0] < 2.0e-2 and errs[1] < 0.7 * errs[0], errs
