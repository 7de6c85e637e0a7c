"""Pins for the oracle's Riemann solvers (SURVEY.md 8(c) pins P2, P3, P6, P7, P8).

None of these re-type the solver formulas: they use conservation (Rankine-Hugoniot), isentropic /
Riemann-invariant relations, symmetry, published star values and hand-computed numbers.
"""
import os

import numpy as np
import pytest

HERE = os.path.dirname(os.path.abspath(__file__))
EXACT, HLLE, HLLC, ROE = 0, 1, 2, 3
ALL = (EXACT, HLLE, HLLC, ROE)


def flux(W, g):
    """Physical Euler flux of a normal-frame primitive state -- definition of the conservation law."""
    rho, vn, v1, v2, P = W
    E = P / (g - 1) + 0.5 * rho * (vn * vn + v1 * v1 + v2 * v2)
    return np.array([rho * vn, rho * vn * vn + P, rho * vn * v1, rho * vn * v2, (E + P) * vn])


def cons(W, g):
    rho, vn, v1, v2, P = W
    return np.array([rho, rho * vn, rho * v1, rho * v2, P / (g - 1) + 0.5 * rho * (vn * vn + v1 * v1 + v2 * v2)])


def rand_state(rng):
    return np.array([rng.uniform(0.5, 2), rng.normal(), rng.normal(), rng.normal(), rng.uniform(0.5, 2)])


# ---- P2: consistency and mirror symmetry ----------------------------------------------------
@pytest.mark.parametrize("solver", ALL)
def test_consistency_RS_W_W_is_physical_flux(oracle, solver):
    rng = np.random.default_rng(1)
    for _ in range(50):
        W = rand_state(rng)
        F, _ = oracle.riemann(solver, W, W, 1.4)
        assert np.allclose(F, flux(W, 1.4), rtol=0, atol=8 * np.finfo(float).eps * np.abs(flux(W, 1.4)).max())


@pytest.mark.parametrize("solver", ALL)
def test_mirror_symmetry(oracle, solver):
    rng = np.random.default_rng(2)
    flip = np.array([1, -1, 1, 1, 1.0])
    for _ in range(50):
        WL, WR = rand_state(rng), rand_state(rng)
        F, _ = oracle.riemann(solver, WL, WR, 5 / 3)
        Fm, _ = oracle.riemann(solver, WR * flip, WL * flip, 5 / 3)
        # x -> -x : scalar fluxes change sign, normal-momentum flux does not
        assert np.allclose(Fm, F * np.array([-1, 1, -1, -1, -1.0]), rtol=1e-11, atol=1e-12)


# ---- P3: exact solver -----------------------------------------------------------------------
def load_toro():
    rows = []
    for line in open(os.path.join(HERE, "golden", "toro_exact_star.txt")):
        if line.strip() and not line.startswith("#"):
            rows.append([float(x) for x in line.split()])
    return rows


@pytest.mark.parametrize("row", load_toro())
def test_exact_star_matches_published_values(oracle, row):
    rl, ul, pl, rr, ur, pr, ps, us, rsl, rsr = row
    WL, WR = [rl, ul, 0, 0, pl], [rr, ur, 0, 0, pr]
    rc, p, u = oracle.exact_star(WL, WR, 1.4)
    assert rc == 0
    assert p == pytest.approx(ps, rel=3e-3 if ps < 0.01 else 2e-5)
    assert u == pytest.approx(us, rel=2e-5, abs=1e-9)


def star_density_by_conservation(WK, p, u, g, side):
    """Density behind the wave that connects WK to the star state (p,u), from physics only:
    shock -> mass+momentum jump conditions; rarefaction -> constant entropy."""
    rK, uK, PK = WK[0], WK[1], WK[4]
    if p > PK:  # Rankine-Hugoniot: mass flux j = (p - PK)/(uK - u) (sign by side), 1/r = 1/rK - (u-uK)/j
        j = (p - PK) / (uK - u) if side == "L" else (p - PK) / (u - uK)  # j > 0
        inv = 1 / rK - (uK - u) / j if side == "L" else 1 / rK - (u - uK) / j
        return 1 / inv
    return rK * (p / PK) ** (1 / g)


@pytest.mark.parametrize("row", load_toro())
def test_exact_star_satisfies_jump_conditions(oracle, row):
    """Independent of the pressure function: each wave must satisfy the full Rankine-Hugoniot
    conditions (mass, momentum AND energy) or, for a rarefaction, carry the Riemann invariant."""
    g = 1.4
    rl, ul, pl, rr, ur, pr, ps, us, rsl, rsr = row
    WL, WR = np.array([rl, ul, 0, 0, pl]), np.array([rr, ur, 0, 0, pr])
    rc, p, u = oracle.exact_star(WL, WR, g)
    for WK, side, rs_pub in ((WL, "L", rsl), (WR, "R", rsr)):
        rs = star_density_by_conservation(WK, p, u, g, side)
        assert rs == pytest.approx(rs_pub, rel=3e-3 if ps < 0.01 else 3e-5)
        Ws = np.array([rs, u, 0, 0, p])
        if p > WK[4]:  # shock: S from mass, then energy jump must hold too
            S = (rs * u - WK[0] * WK[1]) / (rs - WK[0])
            jump = flux(Ws, g) - flux(WK, g) - S * (cons(Ws, g) - cons(WK, g))
            assert np.abs(jump).max() < 1e-9 * max(1.0, np.abs(flux(Ws, g)).max())
        else:  # rarefaction: u +- 2c/(g-1) constant
            cK, cs = np.sqrt(g * WK[4] / WK[0]), np.sqrt(g * p / rs)
            sgn = 1 if side == "L" else -1
            assert u + sgn * 2 * cs / (g - 1) == pytest.approx(WK[1] + sgn * 2 * cK / (g - 1), rel=1e-10, abs=1e-10)


def sample_at(oracle, WL, WR, g, xi):
    """Exact solution at x/t = xi through the oracle's x/t = 0 sampler and Galilean invariance."""
    sh = np.array([0, xi, 0, 0, 0.0])
    rc, W = oracle.exact_sample0(np.asarray(WL) - sh, np.asarray(WR) - sh, g)
    assert rc == 0
    return W + sh


def test_exact_sampler_sod_structure(oracle):
    """Sod: fan head/tail, contact and shock positions (SURVEY P3 list) and the fan interior,
    checked through invariants: inside the fan entropy and u + 2c/(g-1) equal the left state's,
    and u - c = x/t (the defining property of a centred left rarefaction)."""
    g = 1.4
    WL, WR = [1, 0, 0.3, -0.2, 1], [0.125, 0, -0.1, 0.4, 0.1]
    cL = np.sqrt(g)
    for xi in np.linspace(-1.18, -0.08, 12):  # inside the fan (head -1.1832, tail -0.0703)
        W = sample_at(oracle, WL, WR, g, xi)
        c = np.sqrt(g * W[4] / W[0])
        assert W[1] - c == pytest.approx(xi, abs=1e-12)
        assert W[4] / W[0] ** g == pytest.approx(1.0, rel=1e-12)
        assert W[1] + 2 * c / (g - 1) == pytest.approx(2 * cL / (g - 1), rel=1e-12)
        assert (W[2], W[3]) == (0.3, -0.2)
    assert np.allclose(sample_at(oracle, WL, WR, g, -1.19), WL)
    assert np.allclose(sample_at(oracle, WL, WR, g, 1.76), WR)
    a, b = sample_at(oracle, WL, WR, g, 0.92), sample_at(oracle, WL, WR, g, 0.93)  # across the contact
    assert a[0] == pytest.approx(0.42632, rel=2e-5) and b[0] == pytest.approx(0.26557, rel=2e-5)
    assert (a[2], a[3]) == (0.3, -0.2) and (b[2], b[3]) == (-0.1, 0.4)  # transverse velocity is upwinded
    assert sample_at(oracle, WL, WR, g, 1.75)[0] == pytest.approx(0.26557, rel=2e-5)  # shock speed 1.75216


def test_exact_star_is_root_by_bisection(oracle):
    """p* from Newton agrees with a bisection root of u*_L(p) = u*_R(p), where u*_K(p) is built from
    the wave relations in mass-flux form (Godunov's formulation), for random data."""
    g = 1.4
    rng = np.random.default_rng(5)

    def u_from_side(WK, p, side):
        rK, uK, PK = WK[0], WK[1], WK[4]
        cK = np.sqrt(g * PK / rK)
        if p > PK:
            j = np.sqrt(rK * ((g + 1) / 2 * p + (g - 1) / 2 * PK))  # Lagrangian mass flux of a shock
            d = (p - PK) / j
        else:
            d = 2 * cK / (g - 1) * ((p / PK) ** ((g - 1) / (2 * g)) - 1)
        return uK - d if side == "L" else uK + d

    for _ in range(30):
        WL, WR = rand_state(rng), rand_state(rng)
        WL[1], WR[1] = rng.normal() * 0.5, rng.normal() * 0.5
        rc, p, u = oracle.exact_star(WL, WR, g)
        assert rc == 0
        lo, hi = 1e-8, 50.0
        for _ in range(200):
            mid = 0.5 * (lo + hi)
            if u_from_side(WL, mid, "L") - u_from_side(WR, mid, "R") > 0:
                lo = mid
            else:
                hi = mid
        assert p == pytest.approx(0.5 * (lo + hi), rel=1e-10)
        assert u == pytest.approx(u_from_side(WL, p, "L"), abs=1e-10)


# ---- P6: isolated waves ---------------------------------------------------------------------
def test_stationary_contact(oracle):
    g = 1.4
    WL, WR = [2.0, 0, 0.3, -0.1, 1.5], [0.5, 0, 0.3, -0.1, 1.5]
    F, _ = oracle.riemann(HLLC, WL, WR, g)
    assert np.array_equal(F, np.array([0, 1.5, 0, 0, 0]))  # exactly
    for s in (ROE, EXACT):
        F, _ = oracle.riemann(s, WL, WR, g)
        assert np.allclose(F, [0, 1.5, 0, 0, 0], atol=1e-14)
    F, _ = oracle.riemann(HLLE, WL, WR, g)
    assert abs(F[0]) > 0.1  # HLLE smears the contact ("more diffusive")


def test_single_shock_roe_returns_upwind_flux(oracle):
    """A right-moving shock obeying Rankine-Hugoniot seen from a frame where it moves with S>0:
    Roe's flux at x/t=0 is F(W_L) (Roe's property U), so are exact and HLLC to rounding."""
    g = 1.4
    r0, P0, M = 1.0, 1.0, 3.0  # pre-shock state at rest, shock Mach 3
    c0 = np.sqrt(g * P0 / r0)
    S = M * c0
    P1 = P0 * (1 + 2 * g / (g + 1) * (M * M - 1))
    r1 = r0 * ((g + 1) * M * M) / ((g - 1) * M * M + 2)
    u1 = S * (1 - r0 / r1)
    WL, WR = np.array([r1, u1, 0.2, 0, P1]), np.array([r0, 0, 0.2, 0, P0])
    assert np.allclose(flux(WL, g) - flux(WR, g), S * (cons(WL, g) - cons(WR, g)), rtol=1e-12)  # data is a shock
    for s in (ROE, EXACT):
        F, st = oracle.riemann(s, WL, WR, g)
        assert np.allclose(F, flux(WL, g), rtol=1e-11)
        assert st[0] == 0


@pytest.mark.parametrize("solver", ALL)
def test_supersonic_returns_upwind_flux(oracle, solver):
    g = 1.4
    WL, WR = np.array([1.0, 5.0, 0.1, 0.2, 1.0]), np.array([0.8, 5.5, -0.1, 0.0, 0.7])
    F, _ = oracle.riemann(solver, WL, WR, g)
    assert np.allclose(F, flux(WL, g), rtol=1e-12)
    flip = np.array([1, -1, 1, 1, 1.0])
    F, _ = oracle.riemann(solver, WR * flip, WL * flip, g)
    assert np.allclose(F, flux(WL * flip, g), rtol=1e-12)


# ---- P7: weak-jump agreement ("brute force on tiny inputs") ---------------------------------
@pytest.mark.parametrize("solver", (ROE, HLLC))
def test_weak_jump_agrees_with_exact_to_second_order(oracle, solver):
    g = 1.4
    rng = np.random.default_rng(7)
    worst = {}
    for eps in (1e-2, 1e-3, 1e-4):
        m = 0.0
        rs = np.random.default_rng(8)
        for _ in range(50):
            WL = rand_state(rs)
            d = rs.normal(size=5)
            WR = WL + eps * d
            Fe, _ = oracle.riemann(EXACT, WL, WR, g)
            F, _ = oracle.riemann(solver, WL, WR, g)
            m = max(m, np.abs(F - Fe).max() / eps ** 2)
        worst[eps] = m
    # the ratio |F - F_exact| / eps^2 stays bounded as eps -> 0  (first-order agreement would grow as 1/eps)
    assert worst[1e-4] < 30 and worst[1e-4] < 3 * worst[1e-2] + 1


def test_hlle_differs_from_exact_at_first_order_on_contacts(oracle):
    """...whereas HLLE is only first-order close on a pure contact jump (control for the pin above)."""
    g = 1.4
    W = np.array([1.0, 0.1, 0, 0, 1.0])
    r = []
    for eps in (1e-2, 1e-4):
        WR = W + eps * np.array([1, 0, 0, 0, 0.0])
        Fe, _ = oracle.riemann(EXACT, W, WR, g)
        Fh, _ = oracle.riemann(HLLE, W, WR, g)
        r.append(np.abs(Fh - Fe).max() / eps)
    assert r[1] == pytest.approx(r[0], rel=0.1) and r[1] > 0.1


# ---- P8: Roe failure and fallback -----------------------------------------------------------
def golden_hand():
    d = {}
    for line in open(os.path.join(HERE, "golden", "roe_failure_hand.txt")):
        if line.strip() and not line.startswith("#"):
            k, v = line.split()
            d[k] = float(v)
    return d


def test_roe_failure_detected_and_fallback_used(oracle):
    g = 1.4
    hand = golden_hand()
    WL, WR = [1, -2, 0, 0, 0.4], [1, 2, 0, 0, 0.4]
    F, st = oracle.riemann(ROE, WL, WR, g, roe_fallback=1)
    assert st[0] == 1
    assert F[1] == pytest.approx(hand["hlle_mom_flux"], abs=2e-6) and abs(F[0]) < 1e-15 and abs(F[4]) < 1e-14
    Fh, _ = oracle.riemann(HLLE, WL, WR, g)
    assert np.array_equal(F, Fh)
    F, st = oracle.riemann(ROE, WL, WR, g, roe_fallback=3)
    assert st[0] == 1 and F[1] == pytest.approx(hand["exact_mom_flux"], rel=1e-5)
    closed = 0.4 * (1 - 0.2 * 4 / (2 * np.sqrt(0.56))) ** 7  # two-rarefaction closed form
    assert F[1] == pytest.approx(closed, rel=1e-9)
    F2, st = oracle.riemann(ROE, WL, WR, g, roe_fallback=2)
    Fc, _ = oracle.riemann(HLLC, WL, WR, g)
    assert st[0] == 1 and np.array_equal(F2, Fc)
    # mild data: no failure
    _, st = oracle.riemann(ROE, [1, -0.1, 0, 0, 0.4], [1, 0.1, 0, 0, 0.4], g)
    assert st[0] == 0


def test_vacuum_counts_and_falls_back(oracle):
    g = 1.4
    WL, WR = [1, -10, 0, 0, 0.4], [1, 10, 0, 0, 0.4]  # 2(cL+cR)/(g-1) = 7.48 < 20
    F, st = oracle.riemann(EXACT, WL, WR, g)
    assert st[2] == 1
    Fh, _ = oracle.riemann(HLLE, WL, WR, g)
    assert np.array_equal(F, Fh)


def test_fp32_solvers_track_fp64(oracle):
    rng = np.random.default_rng(11)
    for solver in ALL:
        for _ in range(20):
            WL, WR = rand_state(rng), rand_state(rng)
            WL32, WR32 = WL.astype(np.float32), WR.astype(np.float32)
            F64, _ = oracle.riemann(solver, WL32.astype(float), WR32.astype(float), 1.4)
            F32, _ = oracle.riemann(solver, WL32, WR32, 1.4, dtype=np.float32)
            assert np.allclose(F32, F64, rtol=0, atol=3e-5 * np.abs(F64).max())
