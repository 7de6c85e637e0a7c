"""Thin ctypes binding of include/hydro.h (argument marshalling only).

Every step of the path runs in the CUDA kernels of libhydro.so; PyTorch supplies device memory
and streams.  There is no CPU fallback: if the library cannot be built or loaded, importing the
entry points raises.  Names follow the C ABI: hydro_solve, hydro_dt, hydro_min_ghost,
hydro_has_fused, hydro_workspace_bytes, hydro_strerror, HydroPipeline (hydro_pipeline_*).
"""
import ctypes as C
import os

import torch  # loads libcudart before libhydro.so is opened

from . import build as _build

MHM, VL, CTU = 0, 1, 2
EXACT, HLLE, HLLC, ROE = 0, 1, 2, 3
GMINMOD, VANLEER, VANALBADA, HYBRID = 0, 1, 2, 3
PLM, PPM = 0, 1
IMPL_AUTO, IMPL_STAGED, IMPL_FUSED = 0, 1, 2
PS = 16

EXPORTS = ("hydro_solve_f32", "hydro_solve_f64", "hydro_dt_f32", "hydro_dt_f64", "hydro_pipeline_create",
           "hydro_pipeline_destroy", "hydro_pipeline_solve_f32", "hydro_pipeline_solve_f64", "hydro_min_ghost",
           "hydro_solve_grid_f32", "hydro_solve_grid_f64", "hydro_gather_f32", "hydro_gather_f64", "hydro_scatter_f32", "hydro_scatter_f64",
           "hydro_has_fused", "hydro_fused_fits", "hydro_workspace_bytes", "hydro_staged_workspace_bytes", "hydro_strerror",
           "hydro_alu_peak_launch", "hydro_advance_f32", "hydro_advance_f64", "hydro_advance_workspace_bytes", "hydro_fluxfix_f32", "hydro_fluxfix_f64", "hydro_restrict_f32", "hydro_restrict_f64",
           "hydro_flux_accum_f32", "hydro_flux_accum_f64", "hydro_rtvd_solve_f32", "hydro_rtvd_solve_f64", "hydro_rtvd_workspace_bytes",
           "hydro_rtvd_solve_noalloc_f64", "hydro_waf_solve_f32", "hydro_waf_solve_f64")


class HydroOpts(C.Structure):
    _fields_ = [("recon", C.c_int), ("nghost", C.c_int), ("char_limit", C.c_int), ("minmod_coeff", C.c_float),
                ("roe_fallback", C.c_int), ("min_dens", C.c_double), ("min_pres", C.c_double),
                ("status", C.c_void_p), ("workspace", C.c_void_p), ("workspace_bytes", C.c_size_t),
                ("impl", C.c_int), ("max_speed", C.c_void_p), ("cfl", C.c_double),
                ("next_max_speed", C.c_void_p), ("next_norm", C.c_int)]


class HydroError(RuntimeError):
    def __init__(self, code, what):
        super().__init__(f"{what}: {hydro_strerror(code)} (code {code})")
        self.code = code


_lib = None


def lib():
    """Load (building if stale) libhydro.so.  Raises if nvcc / the library is unavailable."""
    global _lib
    if _lib is None:
        path = _build.LIB
        if os.environ.get("HYDRO_NO_BUILD") != "1" or not os.path.exists(path):
            path = _build.build()
        L = C.CDLL(path)
        vp, i, sz = C.c_void_p, C.c_int, C.c_size_t
        for name, ft in (("f32", C.c_float), ("f64", C.c_double)):
            getattr(L, "hydro_solve_" + name).argtypes = [vp, vp, vp, i, ft, ft, ft, i, i, i, C.POINTER(HydroOpts), vp]
            getattr(L, "hydro_dt_" + name).argtypes = [vp, i, i, ft, i, vp, vp]
            getattr(L, "hydro_solve_grid_" + name).argtypes = [vp, vp, i, i, i, i, ft, ft, ft, i, i, i, C.POINTER(HydroOpts), vp]
            getattr(L, "hydro_advance_" + name).argtypes = [vp, i, i, i, i, i, ft, ft, i, i, i, C.POINTER(HydroOpts), vp, sz, vp, vp]
            getattr(L, "hydro_rtvd_solve_" + name).argtypes = [vp, vp, vp, i, ft, ft, ft, i, C.POINTER(HydroOpts), vp]
            getattr(L, "hydro_waf_solve_" + name).argtypes = [vp, vp, vp, i, ft, ft, ft, i, C.POINTER(HydroOpts), vp]
            getattr(L, "hydro_fluxfix_" + name).argtypes = [vp, vp, vp, vp, i, ft, ft, vp]
            getattr(L, "hydro_restrict_" + name).argtypes = [vp, vp, vp, i, vp]
            getattr(L, "hydro_flux_accum_" + name).argtypes = [vp, vp, C.c_longlong, ft, vp]
            getattr(L, "hydro_pipeline_solve_" + name).argtypes = [vp, vp, vp, vp, i, ft, ft, ft, i, i, i,
                                                                   C.POINTER(HydroOpts), vp, vp]
        L.hydro_rtvd_solve_noalloc_f64.argtypes = [vp, vp, vp, i, C.c_double, C.c_double, C.c_double, i, vp, vp]
        L.hydro_pipeline_create.argtypes = [C.POINTER(vp), i, i, i, i]
        L.hydro_pipeline_destroy.argtypes = [vp]
        L.hydro_pipeline_destroy.restype = None
        for name in ("f32", "f64"):
            getattr(L, "hydro_gather_" + name).argtypes = [vp, vp, i, i, i, i, i, vp]
            getattr(L, "hydro_scatter_" + name).argtypes = [vp, vp, i, i, i, vp]
        L.hydro_min_ghost.argtypes = [i, i]
        L.hydro_has_fused.argtypes = [i, i, i, i]
        L.hydro_fused_fits.argtypes = [i, i, i, i]
        L.hydro_workspace_bytes.argtypes = [i, i, i, i]
        L.hydro_workspace_bytes.restype = sz
        L.hydro_staged_workspace_bytes.argtypes = [i, i, i, i]
        L.hydro_staged_workspace_bytes.restype = sz
        L.hydro_alu_peak_launch.argtypes = [i, i, i, i, vp, C.POINTER(C.c_double), vp]
        L.hydro_rtvd_workspace_bytes.argtypes = [i, i]
        L.hydro_rtvd_workspace_bytes.restype = sz
        L.hydro_advance_workspace_bytes.argtypes = [i, i, i, i, i, i, C.POINTER(HydroOpts)]
        L.hydro_advance_workspace_bytes.restype = sz
        L.hydro_strerror.argtypes = [i]
        L.hydro_strerror.restype = C.c_char_p
        _lib = L
    return _lib


def hydro_strerror(code):
    return lib().hydro_strerror(int(code)).decode()


def hydro_min_ghost(scheme, recon=PLM):
    return lib().hydro_min_ghost(scheme, recon)


def hydro_has_fused(dtype, scheme, recon=PLM, riemann=ROE):
    return bool(lib().hydro_has_fused(torch.empty((), dtype=dtype).element_size(), scheme, recon, riemann))


def hydro_fused_fits(dtype, scheme, recon=PLM, nghost=0):
    return bool(lib().hydro_fused_fits(torch.empty((), dtype=dtype).element_size(), scheme, recon, nghost))


def hydro_workspace_bytes(Ng, dtype, scheme, recon=PLM, impl=IMPL_AUTO, nghost=0):
    """Scratch bytes hydro_solve needs: 0 when the fused kernel runs for this ghost width."""
    es = torch.empty((), dtype=dtype).element_size()
    if impl == IMPL_STAGED or (impl == IMPL_AUTO and not lib().hydro_fused_fits(es, scheme, recon, nghost)):
        return lib().hydro_staged_workspace_bytes(Ng, es, scheme, recon)
    return 0


def _workspace(nbytes, device):
    """A fresh caller-owned scratch tensor for the staged path (nothing is cached between calls: two calls on different
    streams must not share scratch; pass workspace= to reuse one)."""
    if nbytes == 0:
        return None
    return torch.empty(nbytes, dtype=torch.uint8, device=device)


def _suffix(t):
    if t.dtype == torch.float32:
        return "f32", C.c_float
    if t.dtype == torch.float64:
        return "f64", C.c_double
    raise TypeError("hydro: dtype must be float32 or float64")


def make_opts(*, recon=PLM, nghost=0, char_limit=0, minmod_coeff=0.0, roe_fallback=0, min_dens=0.0, min_pres=0.0,
              status=None, workspace=None, impl=IMPL_AUTO, max_speed=None, cfl=0.0, next_max_speed=None, next_norm=0):
    o = HydroOpts()
    o.recon, o.nghost, o.char_limit, o.minmod_coeff, o.roe_fallback = recon, nghost, char_limit, minmod_coeff, roe_fallback
    o.min_dens, o.min_pres, o.impl = min_dens, min_pres, impl
    o.max_speed = max_speed.data_ptr() if max_speed is not None else None
    o.cfl = cfl
    o.next_max_speed = next_max_speed.data_ptr() if next_max_speed is not None else None
    o.next_norm = next_norm
    o.status = status.data_ptr() if status is not None else None
    o.workspace = workspace.data_ptr() if workspace is not None else None
    o.workspace_bytes = workspace.numel() * workspace.element_size() if workspace is not None else 0
    return o


def hydro_solve(in_, dt, dh, gamma, scheme=CTU, riemann=ROE, limiter=VANLEER, *, out=None, face_flux=True,
                status=None, stream=None, **optkw):
    """hydro_solve_f32/f64 on CUDA tensors.  in_[Ng,5,S,S,S]; returns (out[Ng,5,16,16,16], face_flux or None).

    face_flux: True -> allocate, False/None -> skip step (5), or a tensor [Ng,9,5,16,16] to fill.
    status: optional int64 CUDA tensor [3], accumulated.  Asynchronous on `stream` (default: current).
    max_speed=<device scalar from hydro_dt>, cfl=<number>: dt is formed on the device and `dt` is ignored.
    """
    if not in_.is_cuda:
        raise ValueError("hydro_solve: `in_` must be a CUDA tensor (host buffers go through HydroPipeline)")
    if not in_.is_contiguous() or in_.dim() != 5 or in_.shape[1] != 5:
        raise ValueError("hydro_solve: in_ must be contiguous [Ng,5,S,S,S]")
    sfx, ft = _suffix(in_)
    Ng, S = in_.shape[0], in_.shape[2]
    g = (S - PS) // 2
    if tuple(in_.shape[2:]) != (S, S, S) or S != PS + 2 * g:
        raise ValueError("hydro_solve: bad padded shape")
    if out is None:
        out = torch.empty((Ng, 5, PS, PS, PS), dtype=in_.dtype, device=in_.device)
    if face_flux is True:
        face_flux = torch.empty((Ng, 9, 5, PS, PS), dtype=in_.dtype, device=in_.device)
    elif face_flux is False:
        face_flux = None
    for t in (out, face_flux):
        if t is not None and (t.dtype != in_.dtype or t.device != in_.device or not t.is_contiguous()):
            raise ValueError("hydro_solve: out / face_flux must match in_ (dtype, device) and be contiguous")
    recon = optkw.get("recon", PLM)
    impl = optkw.get("impl", IMPL_AUTO)
    ws = optkw.pop("workspace", None)
    if ws is None:
        ws = _workspace(hydro_workspace_bytes(Ng, in_.dtype, scheme, recon, impl, g), in_.device)
    o = make_opts(nghost=g, status=status, workspace=ws, **optkw)
    st = (stream or torch.cuda.current_stream(in_.device)).cuda_stream
    with torch.cuda.device(in_.device):
        rc = getattr(lib(), "hydro_solve_" + sfx)(in_.data_ptr(), out.data_ptr(),
                                                  face_flux.data_ptr() if face_flux is not None else None, Ng,
                                                  ft(dt), ft(dh), ft(gamma), scheme, riemann, limiter, C.byref(o), st)
    if rc != 0:
        raise HydroError(rc, "hydro_solve_" + sfx)
    if ws is not None and stream is not None:
        ws.record_stream(stream)  # the kernel may still be using it when the tensor goes back to the allocator
    return out, face_flux


def _stream(t, stream):
    return (stream or torch.cuda.current_stream(t.device)).cuda_stream


def hydro_waf_solve(in_, dt, dh, gamma, order=0, **kw):
    """hydro_waf_solve_f32/f64: one directionally split weighted-average-flux step; arguments as hydro_rtvd_solve."""
    return hydro_rtvd_solve(in_, dt, dh, gamma, order, _entry="hydro_waf_solve_", **kw)


def hydro_rtvd_solve(in_, dt, dh, gamma, order=0, *, out=None, face_flux=True, status=None, workspace=None, stream=None,
                     max_speed=None, cfl=0.0, _entry="hydro_rtvd_solve_"):
    """hydro_rtvd_solve_f32/f64: one directionally split relaxing-TVD step (sweeps x,y,z for order 0; z,y,x for order 1) of
    in_[Ng,5,S,S,S] (ghost width >= 3).  Returns (out, face_flux or None).  workspace: uint8 CUDA tensor of
    hydro_rtvd_workspace_bytes(Ng, precision) (allocated if None)."""
    if not in_.is_cuda or not in_.is_contiguous() or in_.dim() != 5 or in_.shape[1] != 5:
        raise ValueError("hydro_rtvd_solve: in_ must be a contiguous CUDA tensor [Ng,5,S,S,S]")
    sfx, ft = _suffix(in_)
    Ng, S = in_.shape[0], in_.shape[2]
    g = (S - PS) // 2
    if out is None:
        out = torch.empty((Ng, 5, PS, PS, PS), dtype=in_.dtype, device=in_.device)
    if face_flux is True:
        face_flux = torch.empty((Ng, 9, 5, PS, PS), dtype=in_.dtype, device=in_.device)
    elif face_flux is False:
        face_flux = None
    if workspace is None:
        workspace = torch.empty(max(16, lib().hydro_rtvd_workspace_bytes(Ng, in_.element_size())), dtype=torch.uint8, device=in_.device)
    o = make_opts(nghost=g, status=status, workspace=workspace, max_speed=max_speed, cfl=cfl)
    with torch.cuda.device(in_.device):
        rc = getattr(lib(), _entry + sfx)(in_.data_ptr(), out.data_ptr(),
                                                       face_flux.data_ptr() if face_flux is not None else None, Ng, ft(dt), ft(dh),
                                                       ft(gamma), order, C.byref(o), _stream(in_, stream))
    if rc != 0:
        raise HydroError(rc, _entry + sfx)
    if stream is not None:
        workspace.record_stream(stream)
    return out, face_flux


RTVD_NOALLOC_MAX_GROUPS = 4096  # HYDRO_RTVD_NOALLOC_MAX_GROUPS of include/hydro.h


def hydro_rtvd_solve_noalloc(in_, dt, dh, gamma, order=0, *, out, face_flux=None, status=None, stream=None):
    """hydro_rtvd_solve_noalloc_f64: the split relaxing-TVD update of fp64 groups with ghost width 3 through the entry point that
    allocates nothing (scratch in a static device array of the library; at most RTVD_NOALLOC_MAX_GROUPS groups per call; calls
    that overlap on the GPU race).  `out` (and `face_flux`, `status`) are caller tensors: this wrapper allocates nothing either."""
    if not in_.is_cuda or in_.dtype != torch.float64 or not in_.is_contiguous() or in_.dim() != 5 or tuple(in_.shape[1:]) != (5, 22, 22, 22):
        raise ValueError("hydro_rtvd_solve_noalloc: in_ must be a contiguous CUDA float64 tensor [Ng,5,22,22,22]")
    for t in (out, face_flux):
        if t is not None and (t.dtype != in_.dtype or t.device != in_.device or not t.is_contiguous()):
            raise ValueError("hydro_rtvd_solve_noalloc: out / face_flux must match in_ (dtype, device) and be contiguous")
    st = (stream or torch.cuda.current_stream(in_.device)).cuda_stream
    with torch.cuda.device(in_.device):
        rc = lib().hydro_rtvd_solve_noalloc_f64(in_.data_ptr(), out.data_ptr(), face_flux.data_ptr() if face_flux is not None else None,
                                                in_.shape[0], dt, dh, gamma, order,
                                                status.data_ptr() if status is not None else None, st)
    if rc != 0:
        raise HydroError(rc, "hydro_rtvd_solve_noalloc_f64")
    return out, face_flux


def hydro_dt(u, gamma, norm=0, *, max_speed=None, stream=None):
    """hydro_dt_f32/f64: device scalar tensor holding the maximum wave speed over interior cells."""
    if not u.is_cuda or not u.is_contiguous() or u.dim() != 5 or u.shape[1] != 5:
        raise ValueError("hydro_dt: u must be a contiguous CUDA tensor [Ng,5,S,S,S]")
    sfx, ft = _suffix(u)
    Ng, S = u.shape[0], u.shape[2]
    g = (S - PS) // 2
    if max_speed is None:
        max_speed = torch.empty((), dtype=u.dtype, device=u.device)
    st = (stream or torch.cuda.current_stream(u.device)).cuda_stream
    with torch.cuda.device(u.device):
        rc = getattr(lib(), "hydro_dt_" + sfx)(u.data_ptr(), Ng, g, ft(gamma), norm, max_speed.data_ptr(), st)
    if rc != 0:
        raise HydroError(rc, "hydro_dt_" + sfx)
    return max_speed


PEAK_KINDS = {"ffma": 0, "ffma2": 1, "dfma": 2, "fmul_fadd": 3, "ffma_fmnmx": 4, "ffma2_fmnmx": 5, "mufu": 6, "ffma_const": 7,
              "2ffma_shf": 8, "ffma2_shf": 9, "6ffma_sel_shf": 10, "3ffma2_sel_shf": 11, "8ffma_sel_mufu_shf": 12, "4ffma2_sel_mufu_shf": 13}


def hydro_alu_peak_launch(kind, blocks, threads, iters, scratch, *, stream=None):
    """hydro_alu_peak_launch: one launch of a register-resident ALU loop; returns its operation count (FMA = 2)."""
    ops = C.c_double()
    st = (stream or torch.cuda.current_stream(scratch.device)).cuda_stream
    with torch.cuda.device(scratch.device):
        rc = lib().hydro_alu_peak_launch(PEAK_KINDS[kind] if isinstance(kind, str) else kind, blocks, threads, iters,
                                         scratch.data_ptr(), C.byref(ops), st)
    if rc != 0:
        raise HydroError(rc, "hydro_alu_peak_launch")
    return ops.value


def hydro_fluxfix(coarse_out, coarse_flux, fine_flux, faces, dt_c, dh_c, *, stream=None):
    """hydro_fluxfix_f32/f64: in place on coarse_out[Nc,5,16,16,16]; faces: CUDA int32 [n,7]."""
    sfx, ft = _suffix(coarse_out)
    if faces.dtype != torch.int32 or not faces.is_cuda or not faces.is_contiguous():
        raise ValueError("hydro_fluxfix: faces must be a contiguous CUDA int32 tensor [n,7]")
    with torch.cuda.device(coarse_out.device):
        rc = getattr(lib(), "hydro_fluxfix_" + sfx)(coarse_out.data_ptr(), coarse_flux.data_ptr(), fine_flux.data_ptr(),
                                                    faces.data_ptr(), faces.shape[0], ft(dt_c), ft(dh_c), _stream(coarse_out, stream))
    if rc != 0:
        raise HydroError(rc, "hydro_fluxfix_" + sfx)
    return coarse_out


def hydro_restrict(fine_out, coarse_out, rmap, *, stream=None):
    """hydro_restrict_f32/f64: in place on coarse_out; rmap: CUDA int32 [n,5]."""
    sfx, _ = _suffix(coarse_out)
    if rmap.dtype != torch.int32 or not rmap.is_cuda or not rmap.is_contiguous():
        raise ValueError("hydro_restrict: map must be a contiguous CUDA int32 tensor [n,5]")
    with torch.cuda.device(coarse_out.device):
        rc = getattr(lib(), "hydro_restrict_" + sfx)(fine_out.data_ptr(), coarse_out.data_ptr(), rmap.data_ptr(), rmap.shape[0],
                                                     _stream(coarse_out, stream))
    if rc != 0:
        raise HydroError(rc, "hydro_restrict_" + sfx)
    return coarse_out


def hydro_flux_accum(acc, face_flux, w, *, stream=None):
    """hydro_flux_accum_f32/f64: acc += w * face_flux (same shape, contiguous)."""
    sfx, ft = _suffix(acc)
    with torch.cuda.device(acc.device):
        rc = getattr(lib(), "hydro_flux_accum_" + sfx)(acc.data_ptr(), face_flux.data_ptr(), acc.numel(), ft(w), _stream(acc, stream))
    if rc != 0:
        raise HydroError(rc, "hydro_flux_accum_" + sfx)
    return acc


BC_PERIODIC, BC_OUTFLOW = 0, 1


def hydro_gather(grid, nghost, bc=BC_PERIODIC, *, groups=None, stream=None):
    """hydro_gather_f32/f64: padded patch groups [Ng,5,S,S,S] of a CUDA grid [5,Nz,Ny,Nx] (multiples of 16)."""
    if not grid.is_cuda or not grid.is_contiguous() or grid.dim() != 4 or grid.shape[0] != 5:
        raise ValueError("hydro_gather: grid must be a contiguous CUDA tensor [5,Nz,Ny,Nx]")
    sfx, _ = _suffix(grid)
    nz, ny, nx = grid.shape[1:]
    S = PS + 2 * nghost
    Ng = (nx // PS) * (ny // PS) * (nz // PS)
    if groups is None:
        groups = torch.empty((Ng, 5, S, S, S), dtype=grid.dtype, device=grid.device)
    st = (stream or torch.cuda.current_stream(grid.device)).cuda_stream
    with torch.cuda.device(grid.device):
        rc = getattr(lib(), "hydro_gather_" + sfx)(grid.data_ptr(), groups.data_ptr(), nx, ny, nz, nghost, bc, st)
    if rc != 0:
        raise HydroError(rc, "hydro_gather_" + sfx)
    return groups


def hydro_scatter(out, shape, *, grid=None, stream=None):
    """hydro_scatter_f32/f64: interiors out[Ng,5,16,16,16] back into a grid [5,Nz,Ny,Nx] with shape = (Nz,Ny,Nx)."""
    if not out.is_cuda or not out.is_contiguous() or out.dim() != 5 or tuple(out.shape[1:]) != (5, PS, PS, PS):
        raise ValueError("hydro_scatter: out must be a contiguous CUDA tensor [Ng,5,16,16,16]")
    sfx, _ = _suffix(out)
    nz, ny, nx = shape
    if out.shape[0] != (nx // PS) * (ny // PS) * (nz // PS):
        raise ValueError("hydro_scatter: group count does not match the grid shape")
    if grid is None:
        grid = torch.empty((5, nz, ny, nx), dtype=out.dtype, device=out.device)
    st = (stream or torch.cuda.current_stream(out.device)).cuda_stream
    with torch.cuda.device(out.device):
        rc = getattr(lib(), "hydro_scatter_" + sfx)(out.data_ptr(), grid.data_ptr(), nx, ny, nz, st)
    if rc != 0:
        raise HydroError(rc, "hydro_scatter_" + sfx)
    return grid


def hydro_solve_grid(grid, dt, dh, gamma, scheme=CTU, riemann=ROE, limiter=VANLEER, *, bc=BC_PERIODIC, out=None, status=None,
                     stream=None, **optkw):
    """hydro_solve_grid_f32/f64: one update of a uniform CUDA grid [5,Nz,Ny,Nx] in one launch (no gather / scatter).
    Returns the updated grid (`out`, allocated if None; must not be `grid`).  Raises HydroError(HYDRO_E_NOFUSED)
    for the one variant without a grid mode (VL with positivity floors)."""
    if not grid.is_cuda or not grid.is_contiguous() or grid.dim() != 4 or grid.shape[0] != 5:
        raise ValueError("hydro_solve_grid: grid must be a contiguous CUDA tensor [5,Nz,Ny,Nx]")
    sfx, ft = _suffix(grid)
    nz, ny, nx = grid.shape[1:]
    if out is None:
        out = torch.empty_like(grid)
    o = make_opts(status=status, **optkw)
    st = (stream or torch.cuda.current_stream(grid.device)).cuda_stream
    with torch.cuda.device(grid.device):
        rc = getattr(lib(), "hydro_solve_grid_" + sfx)(grid.data_ptr(), out.data_ptr(), nx, ny, nz, bc, ft(dt), ft(dh), ft(gamma),
                                                      scheme, riemann, limiter, C.byref(o), st)
    if rc != 0:
        raise HydroError(rc, "hydro_solve_grid_" + sfx)
    return out


def hydro_advance_workspace_bytes(shape, dtype, scheme, limiter=VANLEER, **optkw):
    """hydro_advance_workspace_bytes for a grid of shape (Nz, Ny, Nx)."""
    o = make_opts(**optkw)
    es = torch.empty((), dtype=dtype).element_size()
    return lib().hydro_advance_workspace_bytes(shape[2], shape[1], shape[0], es, scheme, limiter, C.byref(o))


def hydro_advance(grid, steps, dh, gamma, scheme=CTU, riemann=ROE, limiter=VANLEER, *, cfl=0.5, bc=BC_PERIODIC, status=None,
                  graph=False, workspace=None, elapsed=None, stream=None, **optkw):
    """hydro_advance_f32/f64: `steps` updates of a uniform CUDA grid [5,Nz,Ny,Nx] in place, entirely on the device.
    Returns (grid, t) with t a device fp64 scalar holding the elapsed time (`elapsed` if given: the steps' dt are added).
    workspace: uint8 CUDA tensor of hydro_advance_workspace_bytes(...) (allocated if None).  graph=True captures the whole
    call in a CUDA graph and replays it once (launch-bound small grids)."""
    if not grid.is_cuda or not grid.is_contiguous() or grid.dim() != 4 or grid.shape[0] != 5:
        raise ValueError("hydro_advance: grid must be a contiguous CUDA tensor [5,Nz,Ny,Nx]")
    sfx, ft = _suffix(grid)
    nz, ny, nx = grid.shape[1:]
    o = make_opts(status=status, cfl=cfl, **optkw)
    if workspace is None:
        workspace = torch.empty(max(256, lib().hydro_advance_workspace_bytes(nx, ny, nz, grid.element_size(), scheme, limiter, C.byref(o))),
                                dtype=torch.uint8, device=grid.device)
    t = elapsed if elapsed is not None else torch.zeros((), dtype=torch.float64, device=grid.device)

    def call(st):
        with torch.cuda.device(grid.device):
            rc = getattr(lib(), "hydro_advance_" + sfx)(grid.data_ptr(), nx, ny, nz, bc, steps, ft(dh), ft(gamma), scheme, riemann,
                                                        limiter, C.byref(o), workspace.data_ptr(), workspace.numel(), t.data_ptr(), st)
        if rc != 0:
            raise HydroError(rc, "hydro_advance_" + sfx)

    if graph:
        cg = torch.cuda.CUDAGraph()
        torch.cuda.synchronize(grid.device)
        with torch.cuda.graph(cg):  # capture only records; nothing runs here
            call(torch.cuda.current_stream(grid.device).cuda_stream)
        cg.replay()
    else:
        call(_stream(grid, stream))
    return grid, t


class HydroPipeline:
    """hydro_pipeline_*: host buffers in, host buffers out, chunks streamed over `nstreams` CUDA streams
    (PAPER.md:107, 123).  Tensors passed to solve() are CPU tensors (pinned for real overlap)."""

    def __init__(self, dtype, nghost, groups_per_chunk=256, nstreams=4, device=None):
        self.dtype = dtype
        self.g = nghost
        self.device = torch.device("cuda", torch.cuda.current_device()) if device is None else torch.device(device)
        self._h = C.c_void_p()
        es = torch.empty((), dtype=dtype).element_size()
        with torch.cuda.device(self.device):
            rc = lib().hydro_pipeline_create(C.byref(self._h), es, nghost, groups_per_chunk, nstreams)
        if rc != 0:
            raise HydroError(rc, "hydro_pipeline_create")

    def solve(self, in_, out, face_flux, dt, dh, gamma, scheme=CTU, riemann=ROE, limiter=VANLEER, *, status=None,
              max_speed=None, **optkw):
        """status: CPU int64 tensor [3] or None; max_speed: CPU scalar tensor of in_.dtype or None (receives the
        wave-speed maximum of the updated state)."""
        if in_.is_cuda or out.is_cuda or (face_flux is not None and face_flux.is_cuda):
            raise ValueError("HydroPipeline.solve takes host tensors")
        sfx, ft = _suffix(in_)
        Ng = in_.shape[0]
        o = make_opts(nghost=self.g, **optkw)
        with torch.cuda.device(self.device):
            rc = getattr(lib(), "hydro_pipeline_solve_" + sfx)(
                self._h, in_.data_ptr(), out.data_ptr(), face_flux.data_ptr() if face_flux is not None else None, Ng,
                ft(dt), ft(dh), ft(gamma), scheme, riemann, limiter, C.byref(o),
                status.data_ptr() if status is not None else None,
                max_speed.data_ptr() if max_speed is not None else None)
        if rc != 0:
            raise HydroError(rc, "hydro_pipeline_solve_" + sfx)
        return out, face_flux

    def close(self):
        if self._h:
            lib().hydro_pipeline_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
