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
