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


# ---- two-level (coarse + one refined patch) step: plumbing for the flux fix-up / restriction tests ----
def two_level_lists(origin, N):
    """Index lists for ONE refined coarse patch whose first coarse cell is origin = (ox, oy, oz) (multiples of 8) in a periodic
    N^3 coarse grid: faces[6,7] = (fine_group, dir, fine_side, coarse_group, ci, cj, ck) and rmap[1,5] (see include/hydro.h)."""
    G = N // 16
    gidx = lambda c: ((c[2] // 16) * G + (c[1] // 16)) * G + (c[0] // 16)
    faces = []
    for d in range(3):
        for side in (0, 1):
            c0 = list(origin)
            c0[d] = (origin[d] - 1) % N if side == 0 else (origin[d] + 8) % N
            faces.append([0, d, side, gidx(c0), c0[0] % 16, c0[1] % 16, c0[2] % 16])
    rmap = [[0, gidx(origin), origin[0] % 16, origin[1] % 16, origin[2] % 16]]
    return np.array(faces, np.int32), np.array(rmap, np.int32)


def two_level_step(backend, amr, Uc, Uf, origin, dt, dh_c, gamma, scheme, riemann, limiter, *, recon=0, fix=True, **kw):
    """One step of a periodic coarse grid Uc[5,N,N,N] with one refined patch Uf[5,16,16,16] covering the coarse cells
    origin .. origin+8 (same dt on both levels; fine ghost zones by piecewise-constant injection of the coarse data).
    `backend` supplies hydro_solve, `amr` supplies restrict(fine_out, coarse_out, rmap) and fluxfix(coarse_out, coarse_flux,
    fine_flux, faces, dt, dh_c) -- the oracle module or a CUDA adapter.  Returns (Uc_new, Uf_new)."""
    from oracle import oracle as O  # min_ghost only (a table lookup)
    g = O.min_ghost(scheme, recon)
    N = Uc.shape[1]
    ox, oy, oz = origin
    Gc = wl.grid_to_groups(Uc, g, "periodic")
    up = np.repeat(np.repeat(np.repeat(Uc, 2, 1), 2, 2), 2, 3)
    up[:, 2 * oz:2 * oz + 16, 2 * oy:2 * oy + 16, 2 * ox:2 * ox + 16] = Uf
    upp = np.pad(up, ((0, 0), (g, g), (g, g), (g, g)), mode="wrap")
    S = 16 + 2 * g
    Gf = np.ascontiguousarray(upp[None, :, 2 * oz:2 * oz + S, 2 * oy:2 * oy + S, 2 * ox:2 * ox + S])
    out_c, ff_c, _ = backend.solve(Gc, dt, dh_c, gamma, scheme, riemann, limiter, recon=recon, **kw)
    out_f, ff_f, _ = backend.solve(Gf, dt, 0.5 * dh_c, gamma, scheme, riemann, limiter, recon=recon, **kw)
    faces, rmap = two_level_lists(origin, N)
    out_c = np.ascontiguousarray(out_c)
    amr.restrict(np.ascontiguousarray(out_f), out_c, rmap)
    if fix:
        amr.fluxfix(out_c, np.ascontiguousarray(ff_c), np.ascontiguousarray(ff_f), faces, dt, dh_c)
    return wl.groups_to_grid(out_c, Uc.shape[1:]), out_f[0]
