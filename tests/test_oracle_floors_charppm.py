"""Pins for the two option branches round 1 left unpinned ("What's weak" 5):

  (i)  the density / pressure floors of the conserved -> primitive conversion and the final re-floor
       ("rho <- max(rho, min_dens), P <- max(P, min_pres) applied wherever con->prim is
       evaluated and to the final state (E rebuilt from floored P)"; PAPER.md:48, 50 note the problem);
  (ii) characteristic limiting under PPM (SURVEY c1 S8 + c2 S6): each of the three limited slopes of the
       Colella-Woodward interpolation is projected with the eigenvectors of ITS OWN cell.

Expected values are closed forms in exactly representable numbers (floors) and a NumPy evaluation written here from
the SURVEY formulas (PPM), not from the oracle; the PPM pin is shown to discriminate the plausible mistake
(projecting the neighbours' slopes with the centre cell's eigenvectors).
"""
import numpy as np
import pytest

MHM, VL, CTU = 0, 1, 2
EXACT, HLLE, HLLC, ROE = 0, 1, 2, 3
GMINMOD, VANLEER, VANALBADA, HYBRID = 0, 1, 2, 3
PLM, PPM = 0, 1


def uniform_groups(O, scheme, recon, rho, v, P, gamma, Ng=2):
    g = O.min_ghost(scheme, recon)
    S = 16 + 2 * g
    E = P / (gamma - 1) + 0.5 * rho * (v[0] ** 2 + v[1] ** 2 + v[2] ** 2)
    G = np.empty((Ng, 5, S, S, S))
    for q, val in enumerate((rho, rho * v[0], rho * v[1], rho * v[2], E)):
        G[:, q] = val
    return G


# every number below is a dyadic rational and gamma - 1 = 1/2, so all of the conversion arithmetic is exact in fp64
GAMMA, RHO, V = 1.5, 2.0, (0.5, 0.25, -0.5)
KIN = 0.5 * RHO * (0.25 + 0.0625 + 0.25)  # 0.5625


@pytest.mark.parametrize("scheme", (CTU, MHM, VL))
@pytest.mark.parametrize("recon", (PLM, PPM))
def test_inactive_floors_leave_a_uniform_state_bitwise(oracle, scheme, recon):
    # floors below every value met: nothing may change, although the final state goes through prim -> cons again
    G = uniform_groups(oracle, scheme, recon, RHO, V, 0.75, GAMMA)
    out, ff, st = oracle.hydro_solve(G, 0.125, 1.0, GAMMA, scheme, HLLC, VANLEER, recon=recon, min_dens=0.5, min_pres=0.25)
    g = (G.shape[2] - 16) // 2
    assert np.array_equal(out, G[:, :, g:g + 16, g:g + 16, g:g + 16])
    assert st[1] == 0


@pytest.mark.parametrize("scheme", (CTU, MHM, VL))
@pytest.mark.parametrize("riemann", (ROE, HLLE, HLLC, EXACT))
def test_pressure_floor_closed_form(oracle, scheme, riemann):
    # P = 0.25 everywhere, floor 0.75: every conversion must hand P = 0.75 to the scheme, so
    #  * the stored face fluxes are the physical flux of (rho, v, P_floor): F_mn = rho v_n^2 + 0.75 (consistency P2),
    #  * the uniform fluxes cancel in the update, and the final re-floor rebuilds E = P_floor/(gamma-1) + rho |v|^2 / 2
    #    exactly, with rho and the momenta untouched; P was positive, so status[1] stays 0.
    G = uniform_groups(oracle, scheme, PLM, RHO, V, 0.25, GAMMA)
    out, ff, st = oracle.hydro_solve(G, 0.125, 1.0, GAMMA, scheme, riemann, VANLEER, min_pres=0.75)
    assert np.all(out[:, 0] == RHO)
    for d in range(3):
        assert np.all(out[:, 1 + d] == RHO * V[d])
    assert np.all(out[:, 4] == 0.75 / (GAMMA - 1) + KIN)
    assert st[1] == 0
    Efl = 0.75 / (GAMMA - 1) + KIN
    for d in range(3):
        for s in range(3):
            F = ff[:, 3 * d + s]
            assert np.allclose(F[:, 0], RHO * V[d], rtol=1e-14, atol=0)
            assert np.allclose(F[:, 1 + d], RHO * V[d] ** 2 + 0.75, rtol=1e-14, atol=0)
            assert np.allclose(F[:, 4], (Efl + 0.75) * V[d], rtol=1e-14, atol=0)
    # the same data without the floor keeps P = 0.25 in the momentum flux: the floor is what changed it
    _, ff0, _ = oracle.hydro_solve(G, 0.125, 1.0, GAMMA, scheme, riemann, VANLEER)
    assert np.allclose(ff0[:, 0, 1], RHO * V[0] ** 2 + 0.25, rtol=1e-14, atol=0)


def test_negative_pressure_is_counted_and_floored(oracle):
    # E below the kinetic energy: P = (gamma-1)(E - KIN) = -0.125 < 0.  Without floors the conversions count it
    # (status[1], "negative density / pressure"); with the floor the state leaves with P = floor.
    G = uniform_groups(oracle, CTU, PLM, RHO, V, 0.75, GAMMA, Ng=1)
    G[:, 4] = KIN - 0.25
    out, ff, st = oracle.hydro_solve(G, 0.125, 1.0, GAMMA, CTU, HLLE, VANLEER, min_pres=0.5)
    assert np.all(out[:, 4] == 0.5 / (GAMMA - 1) + KIN)
    # every cell of the padded box is converted once and every interior cell once more at the end: a lower bound
    # the region bookkeeping cannot change; it is the same number for any dt (the count is structural)
    assert st[1] >= G.shape[2] ** 3 + 16 ** 3
    _, _, st2 = oracle.hydro_solve(G, 0.0625, 1.0, GAMMA, CTU, HLLE, VANLEER, min_pres=0.5)
    assert st2[1] == st[1]


def test_density_floor_closed_form(oracle):
    # rho = 0.5 below min_dens = 2: the conversion returns rho = 2 (and velocities m / 2); the final state is rebuilt
    # from those primitives: rho = 2, m unchanged (2 * m/2), E = P/(gamma-1) + 2 |m/2|^2 / 2 with the P the conversion saw,
    # P = (gamma-1)(E - 2 |m/2|^2 / 2)  =>  E unchanged as well.  All dyadic: exact.
    rho0, m = 0.5, np.array([0.5, 0.25, -0.5])
    E0 = 4.0
    G = np.empty((1, 5, 20, 20, 20))
    for q, val in enumerate((rho0, m[0], m[1], m[2], E0)):
        G[:, q] = val
    out, _, st = oracle.hydro_solve(G, 0.0625, 1.0, GAMMA, CTU, HLLC, VANLEER, min_dens=2.0)
    assert np.all(out[:, 0] == 2.0)
    for d in range(3):
        assert np.all(out[:, 1 + d] == m[d])
    assert np.all(out[:, 4] == E0)
    assert st[1] == 0  # rho and P positive: nothing to count


# ---- (ii) PPM with characteristic limiting ---------------------------------------------------------------------
def np_limited(dL, dR, lim, theta=1.5):
    """SURVEY c1, written out: zero at extrema, else the named limiter of (dL, dR, dC)."""
    if dL * dR <= 0:
        return 0.0
    dC = 0.5 * (dL + dR)
    s = 1.0 if dC > 0 else -1.0
    if lim == GMINMOD:
        return s * min(theta * abs(dL), theta * abs(dR), abs(dC))
    if lim == VANLEER:
        return 2 * dL * dR / (dL + dR)
    if lim == VANALBADA:
        return dL * dR * (dL + dR) / (dL * dL + dR * dR)
    return s * min(2 * abs(dL), 2 * abs(dR), abs(dC), abs(2 * dL * dR / (dL + dR)))


def np_char_slope(Wm, W0, Wp, g, lim, Weig):
    """S8: project dL, dR with the left eigenvectors of Weig, limit each characteristic component, project back."""
    rho, c = Weig[0], np.sqrt(g * Weig[4] / Weig[0])
    L = np.array([[0, -0.5 * rho / c, 0, 0, 0.5 / c**2], [1, 0, 0, 0, -1 / c**2], [0, 0, 1, 0, 0], [0, 0, 0, 1, 0],
                  [0, 0.5 * rho / c, 0, 0, 0.5 / c**2]])
    Rm = np.array([[1, -c / rho, 0, 0, c * c], [1, 0, 0, 0, 0], [0, 0, 1, 0, 0], [0, 0, 0, 1, 0], [1, c / rho, 0, 0, c * c]]).T
    aL, aR = L @ (W0 - Wm), L @ (Wp - W0)
    a = np.array([np_limited(aL[k], aR[k], lim) for k in range(5)])
    return Rm @ a


def np_ppm_faces(W5, g, lim, own_eigenvectors=True):
    """S6: Colella-Woodward edge values from the three limited slopes + monotonisation (untraced W-, W+)."""
    e = (lambda k: W5[k]) if own_eigenvectors else (lambda k: W5[2])
    sm = np_char_slope(W5[0], W5[1], W5[2], g, lim, e(1))
    s0 = np_char_slope(W5[1], W5[2], W5[3], g, lim, e(2))
    sp = np_char_slope(W5[2], W5[3], W5[4], g, lim, e(3))
    w0 = W5[2]
    wl = 0.5 * (W5[1] + w0) - (s0 - sm) / 6
    wr = 0.5 * (w0 + W5[3]) - (sp - s0) / 6
    for q in range(5):
        if (wr[q] - w0[q]) * (w0[q] - wl[q]) <= 0:
            wl[q] = wr[q] = w0[q]
        else:
            dd, m = wr[q] - wl[q], w0[q] - 0.5 * (wl[q] + wr[q])
            if 6 * dd * m > dd * dd:
                wl[q] = 3 * w0[q] - 2 * wr[q]
            elif 6 * dd * m < -dd * dd:
                wr[q] = 3 * w0[q] - 2 * wl[q]
    return wl, wr


@pytest.mark.parametrize("lim", (GMINMOD, VANLEER, VANALBADA, HYBRID))
def test_ppm_characteristic_limiting_uses_each_cells_own_eigenvectors(oracle, lim):
    g = 1.4
    rng = np.random.default_rng(100 + lim)
    worst_gap = 0.0
    for _ in range(40):
        # a monotone pencil whose sound speed varies by ~2x across the stencil (rho falls 4x, P rises): the eigenvectors of
        # neighbouring cells differ at O(1), so the choice of eigenvectors shows in the edge values
        x = np.arange(5.0)
        rho = 4.0 * np.exp(-0.35 * x) * (1 + 0.03 * rng.normal(size=5))
        P = 1.0 + 0.3 * x + 0.05 * rng.normal(size=5)
        vn = 0.2 + 0.15 * x + 0.02 * rng.normal(size=5)
        W5 = np.stack([rho, vn, 0.1 * x, -0.05 * x, P], axis=1)
        lo, up = oracle.reconstruct(W5, g, 0.3, recon=PPM, limiter=lim, char_limit=1, trace=False)
        wl, wr = np_ppm_faces(W5.copy(), g, lim, own_eigenvectors=True)
        assert np.allclose(lo, wl, rtol=1e-12, atol=1e-13) and np.allclose(up, wr, rtol=1e-12, atol=1e-13)
        bl, br = np_ppm_faces(W5.copy(), g, lim, own_eigenvectors=False)
        worst_gap = max(worst_gap, np.max(np.abs(np.concatenate([bl - wl, br - wr]))))
    # the mistaken variant (centre-cell eigenvectors for all three slopes) is far outside the tolerance above
    assert worst_gap > 1e-3
