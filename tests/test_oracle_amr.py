"""Pins for the consumer of face_flux: coarse-fine flux fix-up + restriction.

What the mathematics fixes: a finite-volume update is conservative iff every face carries ONE flux.  On a two-level
composite grid the faces between an unrefined coarse cell and a refined patch carry the coarse flux on one side and four
fine fluxes on the other; the fix-up replaces the former by the area mean of the latter, so the composite totals of mass,
momentum and energy change by summation rounding only.  That single property pins the sign sigma, the plane index p = 3 d + s
(including the mid-plane s = 1, the reason hydro_solve stores nine planes), the in-plane order of every direction, the factor
1/4 and the factor dt_c/dh_c at once; without the fix-up the totals drift at O(dt).
"""
import numpy as np
import pytest

from tests.harness import OracleBackend, two_level_lists, two_level_step

MHM, VL, CTU = 0, 1, 2
HLLE, HLLC, ROE = 1, 2, 3


def smooth_state(n, dh, gamma, shift=0.0):
    """Smooth periodic state sampled at the centres of an n^3 grid of spacing dh covering [0, n dh)^3 (box length 1)."""
    x = (np.arange(n) + 0.5) * dh + shift
    Z, Y, X = np.meshgrid(x, x, x, indexing="ij")
    tp = 2 * np.pi
    rho = 1.0 + 0.3 * np.sin(tp * X) * np.cos(tp * Y) + 0.2 * np.sin(tp * (Z + 0.3))
    vx = 0.4 * np.sin(tp * (Y + Z))
    vy = -0.3 * np.cos(tp * (X - Z))
    vz = 0.5 * np.sin(tp * (X + 2 * Y))
    P = 1.0 + 0.25 * np.cos(tp * (X + Y + Z))
    E = P / (gamma - 1) + 0.5 * rho * (vx * vx + vy * vy + vz * vz)
    return np.stack([rho, rho * vx, rho * vy, rho * vz, E])


def composite(origin, N=32, gamma=1.4):
    """Coarse N^3 grid + one refined patch; the covered coarse cells hold the restriction of the fine data."""
    dh = 1.0 / N
    Uc = smooth_state(N, dh, gamma)
    fine = smooth_state(2 * N, dh / 2, gamma)
    ox, oy, oz = origin
    Uf = np.ascontiguousarray(fine[:, 2 * oz:2 * oz + 16, 2 * oy:2 * oy + 16, 2 * ox:2 * ox + 16])
    Uc[:, oz:oz + 8, oy:oy + 8, ox:ox + 8] = Uf.reshape(5, 8, 2, 8, 2, 8, 2).mean(axis=(2, 4, 6))
    return Uc, Uf, dh


# origins chosen so that the six faces meet coarse planes f = 0 (s = 0), f = 8 (s = 1, the mid-plane) and f = 16 (s = 2)
ORIGINS = ((8, 8, 8), (0, 16, 24), (24, 0, 8))


@pytest.mark.parametrize("origin", ORIGINS)
@pytest.mark.parametrize("scheme,riemann", ((CTU, ROE), (MHM, HLLC), (VL, HLLE)))
def test_two_level_conservation(oracle, nthreads, origin, scheme, riemann):
    gamma = 1.4
    Uc, Uf, dh = composite(origin)
    G0 = np.ascontiguousarray(Uc[None])  # any layout: only the maximum over cells is needed
    dt = 0.2 * (dh / 2) / 3.0  # well inside the fine level's CFL limit (wave speeds < 3)
    back = OracleBackend(oracle, nthreads)
    tot0 = Uc.sum(axis=(1, 2, 3), dtype=np.float64)
    new_fix, _ = two_level_step(back, oracle, Uc, Uf, origin, dt, dh, gamma, scheme, riemann, 1)
    new_raw, _ = two_level_step(back, oracle, Uc, Uf, origin, dt, dh, gamma, scheme, riemann, 1, fix=False)
    scale = np.abs(Uc).sum(axis=(1, 2, 3))
    drift_fix = np.abs(new_fix.sum(axis=(1, 2, 3), dtype=np.float64) - tot0) / scale
    drift_raw = np.abs(new_raw.sum(axis=(1, 2, 3), dtype=np.float64) - tot0) / scale
    assert drift_fix.max() < 2e-15, drift_fix       # summation rounding of 32768 cells
    assert drift_raw.max() > 1e-9, drift_raw        # the uncorrected composite is NOT conservative: the pin discriminates
    # only the 6 x 64 coarse cells next to the patch were touched by the fix-up
    changed = np.any(new_fix != new_raw, axis=0)
    assert 0 < changed.sum() <= 6 * 64


def test_fixup_is_exactly_the_flux_mismatch(oracle):
    # hand-built fluxes: coarse flux 1 on every face, fine fluxes 1 + checkerboard eps: the mean over 2 x 2 faces is 1
    # exactly -> no change; fine fluxes 3 everywhere -> U changes by sigma nu (1 - 3) exactly (dyadic numbers)
    faces, _ = two_level_lists((8, 8, 8), 32)
    out = np.zeros((8, 5, 16, 16, 16))
    fc = np.ones((8, 9, 5, 16, 16))
    ii, jj = np.meshgrid(np.arange(16), np.arange(16), indexing="ij")
    ff = (1.0 + 0.25 * (-1.0) ** (ii + jj))[None, None, None] * np.ones((1, 9, 5, 1, 1))
    oracle.fluxfix(out, fc, np.ascontiguousarray(ff), faces, 0.5, 2.0)
    assert not out.any()
    oracle.fluxfix(out, fc, np.full((1, 9, 5, 16, 16), 3.0), faces, 0.5, 2.0)
    vals = np.unique(out)
    assert set(vals.tolist()) == {-0.5, 0.0, 0.5}  # nu = 1/4, F_c - Fbar = -2, sigma = +-1
    assert (out != 0).sum() == 6 * 64 * 5
    # fine group above the cells (fine_side 0): sigma = +1, so those cells got +nu (1 - 3) = -0.5: the x-lower face's cells
    assert np.all(out[0, :, 8:16, 8:16, 7] == -0.5)   # group (0,0,0), layer i = 7
    assert np.all(out[1, :, 8:16, 8:16, 0] == 0.5)    # group gx = 1, layer i = 0: the fine group lies below


def test_uniform_state_identity(oracle, nthreads):
    gamma = 5.0 / 3.0
    Uc = np.empty((5, 32, 32, 32))
    for q, v in enumerate((1.5, 0.75, -0.375, 0.25, 2.5)):
        Uc[q] = v
    Uf = np.ascontiguousarray(Uc[:, :16, :16, :16])
    new_c, new_f = two_level_step(OracleBackend(oracle, nthreads), oracle, Uc, Uf, (8, 16, 0), 0.004, 1 / 32, gamma, CTU, ROE, 1)
    assert np.array_equal(new_c, Uc) and np.array_equal(new_f, Uf)


def test_restriction_of_linear_data_is_exact(oracle):
    # dyadic linear data: the mean of the 8 fine cells is the value at the coarse centre, exactly
    k, j, i = np.meshgrid(np.arange(16), np.arange(16), np.arange(16), indexing="ij")
    fine = np.stack([0.5 * i + 0.25 * j - 0.125 * k + q for q in range(5)])[None].astype(np.float64)
    coarse = np.full((2, 5, 16, 16, 16), -7.0)
    oracle.restrict(fine, coarse, np.array([[0, 1, 8, 0, 8]], np.int32))
    kc, jc, ic = np.meshgrid(np.arange(8), np.arange(8), np.arange(8), indexing="ij")
    for q in range(5):
        expect = 0.5 * (2 * ic + 0.5) + 0.25 * (2 * jc + 0.5) - 0.125 * (2 * kc + 0.5) + q
        assert np.array_equal(coarse[1, q, 8:16, 0:8, 8:16], expect)
    mask = np.ones_like(coarse, bool)
    mask[1, :, 8:16, 0:8, 8:16] = False
    assert np.all(coarse[mask] == -7.0)


def test_flux_accumulation(oracle):
    acc = np.zeros((1, 9, 5, 16, 16))
    a, b = np.full_like(acc, 2.0), np.full_like(acc, 4.0)
    oracle.flux_accum(acc, a, 0.5)
    oracle.flux_accum(acc, b, 0.5)
    assert np.all(acc == 3.0)
