"""Uniform-grid multi-step driver used by both the oracle pins and the GPU parity tests.

Pure plumbing (gather ghosts -> hydro_dt -> hydro_solve -> scatter); `backend` supplies the two
calls, so the same loop drives the CPU oracle and the CUDA library.
"""
import numpy as np

from paper_1103_3373_b200 import workloads as wl


class OracleBackend:
    def __init__(self, O, nthreads=1):
        self.O, self.nthreads = O, nthreads

    def dt(self, G, gamma, norm):
        return self.O.hydro_dt(G, gamma, norm)

    def solve(self, G, dt, dh, gamma, scheme, riemann, limiter, **kw):
        return self.O.hydro_solve(G, dt, dh, gamma, scheme, riemann, limiter, nthreads=self.nthreads, **kw)


def run_grid(backend, U, steps, dh, gamma, scheme, riemann, limiter, *, recon=0, cfl=0.5, bc="periodic",
             norm=0, g=None, on_step=None, fixed_dt=None, **kw):
    """Advance grid U[5,Nz,Ny,Nx] by `steps`; returns (U, t, status_total, dts)."""
    from oracle import oracle as O  # only for min_ghost (a table lookup, no arithmetic)
    g = g or O.min_ghost(scheme, recon)
    t, total, dts = 0.0, np.zeros(8, np.int64), []
    shape = U.shape[1:]
    for s in range(steps):
        G = wl.grid_to_groups(U, g, bc)
        if fixed_dt is None:
            smax = backend.dt(G, gamma, norm)
            dt = float(U.dtype.type(cfl * dh / smax))
        else:
            dt = fixed_dt
        out, ff, st = backend.solve(G, dt, dh, gamma, scheme, riemann, limiter, recon=recon, **kw)
        U = wl.groups_to_grid(out, shape)
        total[:len(st)] += st
        t += dt
        dts.append(dt)
        if on_step:
            on_step(s, U, ff, G, dt)
    return U, t, total, dts


class CudaBackend:
    """The CUDA library behind the same two calls (numpy in / numpy out; device work in libhydro)."""

    def __init__(self, impl=0, device="cuda:0"):
        import torch
        from paper_1103_3373_b200 import binding as B
        self.B, self.torch, self.impl, self.device = B, torch, impl, device

    def dt(self, G, gamma, norm):
        t = self.torch.from_numpy(np.ascontiguousarray(G)).to(self.device)
        return float(self.B.hydro_dt(t, gamma, norm).item())

    def solve(self, G, dt, dh, gamma, scheme, riemann, limiter, **kw):
        torch = self.torch
        t = torch.from_numpy(np.ascontiguousarray(G)).to(self.device)
        status = torch.zeros(3, dtype=torch.int64, device=self.device)
        kw.pop("nthreads", None)
        want_flux = kw.pop("want_flux", True)
        out, ff = self.B.hydro_solve(t, dt, dh, gamma, scheme, riemann, limiter, face_flux=want_flux, status=status,
                                     impl=self.impl, **kw)
        torch.cuda.synchronize()
        return out.cpu().numpy(), (ff.cpu().numpy() if ff is not None else None), status.cpu().numpy()
