"""ctypes front end of the CPU oracle (TEST INFRASTRUCTURE ONLY).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  It never imports the CUDA package.  Arrays are numpy, C-contiguous:
  in_[Ng,5,S,S,S] (z,y,x; x fastest), out[Ng,5,16,16,16], face_flux[Ng,9,5,16,16].
"""
import ctypes as C
import os

import numpy as np

from . import build_oracle

MHM, VL, CTU = 0, 1, 2
EXACT, HLLE, HLLC, ROE = 0, 1, 2, 3
GMINMOD, VANLEER, VANALBADA, HYBRID = 0, 1, 2, 3
PLM, PPM = 0, 1
PS = 16


class _Opts(C.Structure):
    _fields_ = [("recon", C.c_int), ("nghost", C.c_int), ("char_limit", C.c_int),
                ("minmod_coeff", C.c_double), ("roe_fallback", C.c_int),
                ("min_dens", C.c_double), ("min_pres", C.c_double),
                ("status", C.POINTER(C.c_longlong)), ("nthreads", C.c_int)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build_oracle.build())
        dp, fp, ip, lp = (C.POINTER(C.c_double), C.POINTER(C.c_float), C.c_int, C.POINTER(C.c_longlong))
        _lib.oracle_hydro_solve_f64.argtypes = [dp, dp, dp, ip, C.c_double, C.c_double, C.c_double, ip, ip, ip,
                                                C.POINTER(_Opts)]
        _lib.oracle_hydro_solve_f32.argtypes = [fp, fp, fp, ip, C.c_float, C.c_float, C.c_float, ip, ip, ip,
                                                C.POINTER(_Opts)]
        _lib.oracle_hydro_dt_f64.argtypes = [dp, ip, ip, C.c_double, ip]
        _lib.oracle_hydro_dt_f64.restype = C.c_double
        _lib.oracle_hydro_dt_f32.argtypes = [fp, ip, ip, C.c_float, ip]
        _lib.oracle_hydro_dt_f32.restype = C.c_float
        _lib.oracle_riemann_f64.argtypes = [ip, dp, dp, C.c_double, ip, dp, lp]
        _lib.oracle_riemann_f32.argtypes = [ip, fp, fp, C.c_float, ip, fp, lp]
        _lib.oracle_exact_star_f64.argtypes = [dp, dp, C.c_double, dp, dp]
        _lib.oracle_exact_sample0_f64.argtypes = [dp, dp, C.c_double, dp]
        _lib.oracle_limited_slope_f64.argtypes = [C.c_double, C.c_double, ip, C.c_double]
        _lib.oracle_limited_slope_f64.restype = C.c_double
        _lib.oracle_reconstruct_f64.argtypes = [dp, C.c_double, C.c_double, ip, ip, ip, C.c_double, ip, dp, dp]
        _lib.oracle_eig_project_f64.argtypes = [dp, C.c_double, dp, dp]
        _lib.oracle_eig_expand_f64.argtypes = [dp, C.c_double, dp, dp]
        _lib.oracle_min_ghost.argtypes = [ip, ip]
    return _lib


def _ptr(a, ct):
    return a.ctypes.data_as(C.POINTER(ct))


def min_ghost(scheme, recon=PLM):
    return lib().oracle_min_ghost(scheme, recon)


def hydro_solve(in_, dt, dh, gamma, scheme=CTU, riemann=ROE, limiter=VANLEER, *, recon=PLM, nghost=0,
                char_limit=0, minmod_coeff=1.5, roe_fallback=1, min_dens=0.0, min_pres=0.0,
                want_flux=True, nthreads=1):
    """One update of Ng padded patch groups.  Returns (out, face_flux or None, status[8])."""
    L = lib()
    in_ = np.ascontiguousarray(in_)
    assert in_.dtype in (np.float32, np.float64) and in_.ndim == 5 and in_.shape[1] == 5
    Ng, S = in_.shape[0], in_.shape[2]
    g = (S - PS) // 2
    assert in_.shape[2:] == (S, S, S) and S == PS + 2 * g
    if nghost:
        assert nghost == g
    out = np.empty((Ng, 5, PS, PS, PS), in_.dtype)
    ff = np.empty((Ng, 9, 5, PS, PS), in_.dtype) if want_flux else None
    status = np.zeros(8, np.int64)
    o = _Opts(recon, g, char_limit, minmod_coeff, roe_fallback, min_dens, min_pres,
              _ptr(status, C.c_longlong), nthreads)
    if in_.dtype == np.float64:
        ct, fn = C.c_double, L.oracle_hydro_solve_f64
    else:
        ct, fn = C.c_float, L.oracle_hydro_solve_f32
    rc = fn(_ptr(in_, ct), _ptr(out, ct), _ptr(ff, ct) if want_flux else None, Ng, dt, dh, gamma,
            scheme, riemann, limiter, C.byref(o))
    if rc != 0:
        raise ValueError(f"oracle_hydro_solve rc={rc}")
    return out, ff, status


def hydro_dt(u, gamma, norm=0):
    """Maximum wave speed over the interior cells of u[Ng,5,S,S,S]."""
    u = np.ascontiguousarray(u)
    Ng, S = u.shape[0], u.shape[2]
    g = (S - PS) // 2
    if u.dtype == np.float64:
        return float(lib().oracle_hydro_dt_f64(_ptr(u, C.c_double), Ng, g, gamma, norm))
    return float(lib().oracle_hydro_dt_f32(_ptr(u, C.c_float), Ng, g, gamma, norm))


def riemann(solver, WL, WR, gamma, roe_fallback=1, dtype=np.float64):
    """Flux of one normal-frame Riemann problem; returns (F[5], status[8])."""
    WL = np.ascontiguousarray(WL, dtype)
    WR = np.ascontiguousarray(WR, dtype)
    F = np.zeros(5, dtype)
    st = np.zeros(8, np.int64)
    if dtype == np.float64:
        lib().oracle_riemann_f64(solver, _ptr(WL, C.c_double), _ptr(WR, C.c_double), gamma, roe_fallback,
                                 _ptr(F, C.c_double), _ptr(st, C.c_longlong))
    else:
        lib().oracle_riemann_f32(solver, _ptr(WL, C.c_float), _ptr(WR, C.c_float), gamma, roe_fallback,
                                 _ptr(F, C.c_float), _ptr(st, C.c_longlong))
    return F, st


def exact_star(WL, WR, gamma):
    WL = np.ascontiguousarray(WL, np.float64)
    WR = np.ascontiguousarray(WR, np.float64)
    p, u = C.c_double(), C.c_double()
    rc = lib().oracle_exact_star_f64(_ptr(WL, C.c_double), _ptr(WR, C.c_double), gamma, C.byref(p), C.byref(u))
    return rc, p.value, u.value


def exact_sample0(WL, WR, gamma):
    WL = np.ascontiguousarray(WL, np.float64)
    WR = np.ascontiguousarray(WR, np.float64)
    W = np.zeros(5)
    rc = lib().oracle_exact_sample0_f64(_ptr(WL, C.c_double), _ptr(WR, C.c_double), gamma, _ptr(W, C.c_double))
    return rc, W


def limited_slope(dL, dR, limiter, theta=1.5):
    return lib().oracle_limited_slope_f64(dL, dR, limiter, theta)


def reconstruct(W5, gamma, nu, recon=PLM, limiter=VANLEER, char_limit=0, theta=1.5, trace=True):
    """Face values (W_lo, W_up) of the middle cell of a 5-cell normal-frame pencil W5[5,5]."""
    W5 = np.ascontiguousarray(W5, np.float64)
    lo, up = np.zeros(5), np.zeros(5)
    lib().oracle_reconstruct_f64(_ptr(W5, C.c_double), gamma, nu, recon, limiter, char_limit, theta, int(trace),
                                 _ptr(lo, C.c_double), _ptr(up, C.c_double))
    return lo, up


def eig_project(W, gamma, d):
    W = np.ascontiguousarray(W, np.float64)
    d = np.ascontiguousarray(d, np.float64)
    a = np.zeros(5)
    lib().oracle_eig_project_f64(_ptr(W, C.c_double), gamma, _ptr(d, C.c_double), _ptr(a, C.c_double))
    return a


def eig_expand(W, gamma, a):
    W = np.ascontiguousarray(W, np.float64)
    a = np.ascontiguousarray(a, np.float64)
    d = np.zeros(5)
    lib().oracle_eig_expand_f64(_ptr(W, C.c_double), gamma, _ptr(a, C.c_double), _ptr(d, C.c_double))
    return d


# ---- consumer of face_flux (oracle/amr_oracle.cpp): coarse-fine flux fix-up and restriction, SURVEY.md 8(f)-3 ----
def _amr_fn(name, dtype):
    L = lib()
    fn = getattr(L, f"oracle_{name}_{'f64' if dtype == np.float64 else 'f32'}")
    fn.restype = None
    return fn, (C.c_double if dtype == np.float64 else C.c_float)


def fluxfix(coarse_out, coarse_flux, fine_flux, faces, dt_c, dh_c):
    """In place on coarse_out[Nc,5,16,16,16]: U += sigma (dt_c/dh_c) (F_c - mean of the 4 fine fluxes) for every
    coarse-fine face listed in faces[n,7] = (fine_group, dir, fine_side, coarse_group, ci, cj, ck) (int32)."""
    faces = np.ascontiguousarray(faces, np.int32).reshape(-1, 7)
    assert coarse_out.flags.c_contiguous and coarse_flux.flags.c_contiguous and fine_flux.flags.c_contiguous
    fn, ct = _amr_fn("fluxfix", coarse_out.dtype.type)
    fn.argtypes = [C.POINTER(ct), C.POINTER(ct), C.POINTER(ct), C.POINTER(C.c_int), C.c_int, ct, ct]
    fn(_ptr(coarse_out, ct), _ptr(coarse_flux, ct), _ptr(fine_flux, ct), _ptr(faces, C.c_int), len(faces), dt_c, dh_c)
    return coarse_out


def restrict(fine_out, coarse_out, rmap):
    """In place on coarse_out: every fine group of rmap[n,5] = (fine_group, coarse_group, pi, pj, pk) replaces the 8^3
    coarse cells starting at (pi, pj, pk) by the means of its 2x2x2 fine cells."""
    rmap = np.ascontiguousarray(rmap, np.int32).reshape(-1, 5)
    assert coarse_out.flags.c_contiguous and fine_out.flags.c_contiguous
    fn, ct = _amr_fn("restrict", coarse_out.dtype.type)
    fn.argtypes = [C.POINTER(ct), C.POINTER(ct), C.POINTER(C.c_int), C.c_int]
    fn(_ptr(fine_out, ct), _ptr(coarse_out, ct), _ptr(rmap, C.c_int), len(rmap))
    return coarse_out


def flux_accum(acc, ff, w):
    """acc += w * ff (dt-weighted time average of the fine fluxes over sub-steps)."""
    fn, ct = _amr_fn("flux_accum", acc.dtype.type)
    fn.argtypes = [C.POINTER(ct), C.POINTER(ct), C.c_longlong, ct]
    fn(_ptr(acc, ct), _ptr(np.ascontiguousarray(ff), ct), acc.size, w)
    return acc


# ---- directionally split relaxing TVD (oracle/rtvd_oracle.cpp), SURVEY.md 8(f)-4 ----
RTVD = 3


def rtvd_solve(in_, dt, dh, gamma, order=0, want_flux=True, nthreads=1):
    """One split RTVD step (sweeps x,y,z for order 0; z,y,x for order 1) of Ng padded groups (g >= 3).
    Returns (out, face_flux or None, status[8])."""
    in_ = np.ascontiguousarray(in_)
    Ng, S = in_.shape[0], in_.shape[2]
    g = (S - PS) // 2
    out = np.empty((Ng, 5, PS, PS, PS), in_.dtype)
    ff = np.empty((Ng, 9, 5, PS, PS), in_.dtype) if want_flux else None
    status = np.zeros(8, np.int64)
    if in_.dtype == np.float64:
        ct, fn = C.c_double, lib().oracle_rtvd_solve_f64
    else:
        ct, fn = C.c_float, lib().oracle_rtvd_solve_f32
    fn.argtypes = [C.POINTER(ct), C.POINTER(ct), C.POINTER(ct), C.c_int, C.c_int, ct, ct, ct, C.c_int, C.POINTER(C.c_longlong), C.c_int]
    rc = fn(_ptr(in_, ct), _ptr(out, ct), _ptr(ff, ct) if want_flux else None, Ng, g, dt, dh, gamma, order,
            _ptr(status, C.c_longlong), nthreads)
    if rc != 0:
        raise ValueError(f"oracle_rtvd_solve rc={rc}")
    return out, ff, status


# ---- directionally split weighted average flux (oracle/waf_oracle.cpp), SURVEY.md 8(f)-4 ----
def waf_solve(in_, dt, dh, gamma, order=0, want_flux=True, nthreads=1):
    """One split WAF step (sweeps x,y,z for order 0; z,y,x for order 1) of Ng padded groups (g >= 3).
    Returns (out, face_flux or None, status[8])."""
    in_ = np.ascontiguousarray(in_)
    Ng, S = in_.shape[0], in_.shape[2]
    g = (S - PS) // 2
    out = np.empty((Ng, 5, PS, PS, PS), in_.dtype)
    ff = np.empty((Ng, 9, 5, PS, PS), in_.dtype) if want_flux else None
    status = np.zeros(8, np.int64)
    if in_.dtype == np.float64:
        ct, fn = C.c_double, lib().oracle_waf_solve_f64
    else:
        ct, fn = C.c_float, lib().oracle_waf_solve_f32
    fn.argtypes = [C.POINTER(ct), C.POINTER(ct), C.POINTER(ct), C.c_int, C.c_int, ct, ct, ct, C.c_int, C.POINTER(C.c_longlong), C.c_int]
    rc = fn(_ptr(in_, ct), _ptr(out, ct), _ptr(ff, ct) if want_flux else None, Ng, g, dt, dh, gamma, order,
            _ptr(status, C.c_longlong), nthreads)
    if rc != 0:
        raise ValueError(f"oracle_waf_solve rc={rc}")
    return out, ff, status


def max_threads():
    return int(lib().oracle_max_threads())
