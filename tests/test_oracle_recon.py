"""Pins for limiters, eigenvectors, PLM/PPM and characteristic tracing (pin P4).

PAPER.md:48 names the limiters and PLM/PPM; PAPER.md:39,46 the characteristic tracing of CTU.
Checks are hand values, defining properties (TVD bounds, exactness on polynomials) and the
single-wave closed form -- none re-types the oracle's formulas.
"""
import numpy as np
import pytest

GMINMOD, VANLEER, VANALBADA, HYBRID = 0, 1, 2, 3
LIMS = (GMINMOD, VANLEER, VANALBADA, HYBRID)
PLM, PPM = 0, 1


# ---- limiters -------------------------------------------------------------------------------
def test_limiter_hand_values(oracle):
    # dL = 1, dR = 3 (dC = 2): worked by hand from the definitions in Toro ch. 13/14
    assert oracle.limited_slope(1, 3, GMINMOD, 1.5) == pytest.approx(1.5)   # min(1.5, 4.5, 2)
    assert oracle.limited_slope(1, 3, GMINMOD, 1.0) == pytest.approx(1.0)   # plain minmod
    assert oracle.limited_slope(1, 3, GMINMOD, 2.0) == pytest.approx(2.0)   # MC: min(2, 6, 2)
    assert oracle.limited_slope(1, 3, VANLEER) == pytest.approx(1.5)        # harmonic mean 2*3/4
    assert oracle.limited_slope(1, 3, VANALBADA) == pytest.approx(1.2)      # 3*4/10
    assert oracle.limited_slope(1, 3, HYBRID) == pytest.approx(1.5)         # min(2, 6, 2, 1.5)
    assert oracle.limited_slope(1, 9, HYBRID) == pytest.approx(1.8)         # min(2, 18, 5, 1.8)
    assert oracle.limited_slope(1, 1.2, HYBRID) == pytest.approx(2 * 1.2 / 2.2)


@pytest.mark.parametrize("lim", LIMS)
def test_limiter_properties(oracle, lim):
    rng = np.random.default_rng(lim)
    for _ in range(200):
        a, b = rng.normal(), rng.normal()
        s = oracle.limited_slope(a, b, lim, 1.5)
        assert s == pytest.approx(oracle.limited_slope(b, a, lim, 1.5), rel=1e-14, abs=0)   # symmetric
        assert s == pytest.approx(-oracle.limited_slope(-a, -b, lim, 1.5), rel=1e-14, abs=0)  # odd
        if a * b <= 0:
            assert s == 0.0                                     # no new extrema
        else:
            assert 0 < s / a <= 2 + 1e-14 and 0 < s / b <= 2 + 1e-14   # Sweby/TVD region
    assert oracle.limited_slope(0.7, 0.7, lim, 1.5) == pytest.approx(0.7)  # linear data reproduced
    assert oracle.limited_slope(0.0, 1.0, lim, 1.5) == 0.0                  # tie-break S19
    assert oracle.limited_slope(-0.7, -0.7, lim, 1.5) == pytest.approx(-0.7)


# ---- eigenvectors ---------------------------------------------------------------------------
def jacobian(W, g):
    """Primitive-variable Jacobian A(W) of the 1-D Euler equations in (rho, vn, vt1, vt2, P)."""
    rho, vn, _, _, P = W
    A = np.eye(5) * vn
    A[0, 1] = rho
    A[1, 4] = 1 / rho
    A[4, 1] = g * P
    return A


def test_eigensystem_diagonalises_the_jacobian(oracle):
    g = 5 / 3
    W = np.array([1.3, 0.4, -0.2, 0.7, 0.9])
    c = np.sqrt(g * W[4] / W[0])
    lam = [W[1] - c, W[1], W[1], W[1], W[1] + c]
    A = jacobian(W, g)
    Rm = np.array([oracle.eig_expand(W, g, np.eye(5)[k]) for k in range(5)]).T   # columns R_k
    Lm = np.array([oracle.eig_project(W, g, np.eye(5)[k]) for k in range(5)]).T  # L e_k = column k
    assert np.allclose(Lm @ Rm, np.eye(5), atol=1e-14)
    assert np.allclose(A @ Rm, Rm @ np.diag(lam), atol=1e-14)


# ---- P4: single-wave exactness of the traced states -----------------------------------------
def pencil_from_slope(W0, slope):
    """5-cell normal-frame pencil with exactly linear data of the given slope vector."""
    return np.array([W0 + s * slope for s in (-2, -1, 0, 1, 2)])


@pytest.mark.parametrize("lim", LIMS)
@pytest.mark.parametrize("wave", range(5))
def test_plm_trace_single_wave(oracle, lim, wave):
    g = 1.4
    for vn in (0.3, -0.4, 2.0, -2.0):  # subsonic both ways and supersonic both ways
        W0 = np.array([1.1, vn, 0.2, -0.3, 0.8])
        c = np.sqrt(g * W0[4] / W0[0])
        lam = [vn - c, vn, vn, vn, vn + c][wave]
        Rk = oracle.eig_expand(W0, g, np.eye(5)[wave])
        a, nu = 1e-3, 0.37
        lo, up = oracle.reconstruct(pencil_from_slope(W0, a * Rk), g, nu, PLM, lim, 0, 1.5, True)
        # Approaching wave: the face average over its domain of dependence (closed form, P4).
        # Receding wave: reading S5 (reference-state form, approaching waves only) leaves the
        # reference state, i.e. the average over the domain of the fastest approaching speed.
        lam_up = lam if lam > 0 else max(vn + c, 0)
        lam_lo = lam if lam < 0 else min(vn - c, 0)
        exp_up = W0 + 0.5 * (1 - nu * lam_up) * a * Rk
        exp_lo = W0 - 0.5 * (1 + nu * lam_lo) * a * Rk
        assert np.allclose(up, exp_up, rtol=0, atol=1e-15)
        assert np.allclose(lo, exp_lo, rtol=0, atol=1e-15)
        # characteristic limiting gives the same slope for linear data
        lo2, up2 = oracle.reconstruct(pencil_from_slope(W0, a * Rk), g, nu, PLM, lim, 1, 1.5, True)
        assert np.allclose(up2, exp_up, atol=1e-15) and np.allclose(lo2, exp_lo, atol=1e-15)


def parabola_cell_averages(a0, a1, a2, n=5):
    """Cell averages over [s-1/2, s+1/2], s=-2..2, of q(x) = a0 + a1 x + a2 x^2."""
    s = np.arange(n) - n // 2
    return a0 + a1 * s + a2 * (s * s + 1 / 12)


def test_ppm_faces_exact_for_parabola_and_traced_average(oracle):
    """PPM with a non-clipping limiter (gminmod theta=2 picks the centred slope on smooth monotone
    data) reproduces a parabola: face values are its point values, and the traced state of a single
    wave is the parabola's average over the last/first nu*|lam| of the cell (closed form, P4)."""
    g = 1.4
    for wave, vn in ((4, 0.3), (0, 0.3), (1, 0.5), (1, -0.5), (4, -2.0), (0, 2.0)):
        W0 = np.array([1.1, vn, 0.2, -0.3, 0.8])
        c = np.sqrt(g * W0[4] / W0[0])
        lam = [vn - c, vn, vn, vn, vn + c][wave]
        Rk = oracle.eig_expand(W0, g, np.eye(5)[wave])
        a1, a2 = 1e-3, 1.5e-4  # monotone over the stencil: |a1| > 4|a2|
        q = parabola_cell_averages(0.0, a1, a2)
        pencil = np.array([W0 + qi * Rk for qi in q]) - q[2] * Rk  # middle cell average == W0
        off = -q[2]

        def par(x):
            return off + a1 * x + a2 * x * x

        lo, up = oracle.reconstruct(pencil, g, 0.0, PPM, GMINMOD, 0, 2.0, False)
        assert np.allclose(up, W0 + par(0.5) * Rk, atol=1e-16 + 1e-13 * abs(a1))
        assert np.allclose(lo, W0 + par(-0.5) * Rk, atol=1e-16 + 1e-13 * abs(a1))
        nu = 0.43

        def avg(x0, x1):  # exact average of the parabola over [x0, x1]
            return off + a1 * (x0 + x1) / 2 + a2 * (x0 * x0 + x0 * x1 + x1 * x1) / 3

        lo, up = oracle.reconstruct(pencil, g, nu, PPM, GMINMOD, 0, 2.0, True)
        s_up = nu * (lam if lam > 0 else max(vn + c, 0))  # receding wave: reference state (S5)
        s_lo = nu * (lam if lam < 0 else min(vn - c, 0))
        exp_up = W0 + (avg(0.5 - s_up, 0.5) if s_up > 0 else par(0.5)) * Rk
        exp_lo = W0 + (avg(-0.5, -0.5 - s_lo) if s_lo < 0 else par(-0.5)) * Rk
        assert np.allclose(up, exp_up, atol=1e-15)
        assert np.allclose(lo, exp_lo, atol=1e-15)


def test_ppm_monotonised_at_extremum_and_steep_gradient(oracle):
    g = 1.4
    base = np.array([1.0, 0.0, 0.0, 0.0, 1.0])
    e0 = np.eye(5)[0]
    # local maximum in rho -> flat
    pencil = np.array([base + r * e0 for r in (0.0, 0.1, 0.3, 0.1, 0.0)])
    lo, up = oracle.reconstruct(pencil, g, 0.0, PPM, VANLEER, 0, 1.5, False)
    assert lo[0] == 1.3 and up[0] == 1.3
    # monotone profile: face values stay within neighbouring cell values, parabola has no interior extremum
    rng = np.random.default_rng(3)
    for _ in range(200):
        r = np.cumsum(rng.uniform(0, 1, 5))
        pencil = np.array([base + ri * e0 for ri in r])
        lo, up = oracle.reconstruct(pencil, g, 0.0, PPM, VANLEER, 0, 1.5, False)
        w0 = pencil[2][0]
        assert pencil[1][0] - 1e-14 <= lo[0] <= w0 <= up[0] <= pencil[3][0] + 1e-14
        D, W6 = up[0] - lo[0], 6 * (w0 - 0.5 * (lo[0] + up[0]))
        assert abs(W6) <= abs(D) * (1 + 1e-12)  # CW84 monotonicity constraint


def test_characteristic_limiting_decouples_waves(oracle):
    """char_limit=1: a jump that is smooth in one family and an extremum in another keeps the smooth
    family's slope (primitive limiting would clip components that mix both)."""
    g = 1.4
    W0 = np.array([1.0, 0.2, 0.0, 0.0, 1.0])
    R1, R5 = oracle.eig_expand(W0, g, np.eye(5)[0]), oracle.eig_expand(W0, g, np.eye(5)[4])
    a = 1e-3
    # acoustic family 5: linear (slope a); acoustic family 1: extremum (+b on both sides)
    b = 0.6e-3
    pencil = np.array([W0 + s * a * R5 + abs(s) * b * R1 for s in (-2, -1, 0, 1, 2)])
    lo, up = oracle.reconstruct(pencil, g, 0.0, PLM, VANLEER, 1, 1.5, False)
    assert np.allclose(up - W0, 0.5 * a * R5, atol=1e-15)
    assert np.allclose(lo - W0, -0.5 * a * R5, atol=1e-15)
    lo_p, up_p = oracle.reconstruct(pencil, g, 0.0, PLM, VANLEER, 0, 1.5, False)
    assert not np.allclose(up_p - W0, 0.5 * a * R5, atol=1e-7)
