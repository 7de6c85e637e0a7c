"""Seeded synthetic inputs and uniform-grid plumbing shared by tests, bench.py and smoke().

This module holds NONE of the method's arithmetic: it only builds initial conditions (primitive
fields -> the conserved 5-vector the paper's solver consumes) and moves cells
between an N^3 SoA grid and padded patch groups (the paper's CPU "preparation"/"closing" steps,
PAPER.md:127, for the trivial uniform-mesh case).  It imports neither the CUDA binding nor the
oracle.  Recipes: DESIGN.md "Input recipe" (configs C1-C5 of BASELINE.json / SURVEY.md 8(d)).

Layouts: grid U[5, Nz, Ny, Nx] (x fastest); groups in_[Ng, 5, S, S, S], S = 16 + 2g;
group index n = (gz * ngy + gy) * ngx + gx.
"""
import numpy as np

PS = 16  # interior cells per side of a patch group


# ------------------------------------------------------------------------------------------
# primitive -> conserved (input construction only)
def prim_to_cons(rho, vx, vy, vz, P, gamma):
    E = P / (gamma - 1.0) + 0.5 * rho * (vx * vx + vy * vy + vz * vz)
    return np.stack([rho, rho * vx, rho * vy, rho * vz, E]).astype(rho.dtype)


# ------------------------------------------------------------------------------------------
# uniform grid <-> patch groups
def grid_to_groups(U, g, bc="periodic"):
    """Gather padded patch groups from U[5,Nz,Ny,Nx].  bc: 'periodic' or 'outflow' (zero-gradient)."""
    assert U.ndim == 4 and U.shape[0] == 5
    nz, ny, nx = (s // PS for s in U.shape[1:])
    assert (nz * PS, ny * PS, nx * PS) == U.shape[1:]
    mode = {"periodic": "wrap", "outflow": "edge"}[bc]
    Up = np.pad(U, ((0, 0), (g, g), (g, g), (g, g)), mode=mode)
    S = PS + 2 * g
    out = np.empty((nz * ny * nx, 5, S, S, S), U.dtype)
    n = 0
    for gz in range(nz):
        for gy in range(ny):
            for gx in range(nx):
                out[n] = Up[:, gz * PS:gz * PS + S, gy * PS:gy * PS + S, gx * PS:gx * PS + S]
                n += 1
    return out


def groups_to_grid(out, shape):
    """Scatter out[Ng,5,16,16,16] back to a grid U[5,Nz,Ny,Nx] with shape=(Nz,Ny,Nx)."""
    nz, ny, nx = (s // PS for s in shape)
    U = np.empty((5,) + tuple(shape), out.dtype)
    n = 0
    for gz in range(nz):
        for gy in range(ny):
            for gx in range(nx):
                U[:, gz * PS:(gz + 1) * PS, gy * PS:(gy + 1) * PS, gx * PS:(gx + 1) * PS] = out[n]
                n += 1
    return U


# ------------------------------------------------------------------------------------------
# C1: Sod shock tube along `axis` (0=x,1=y,2=z) on an N^3 grid, dh = 1/N (BASELINE.json configs[0])
def sod_grid(N=32, axis=0, gamma=1.4, dtype=np.float64):
    x = (np.arange(N) + 0.5) / N
    left = x < 0.5
    shape = [1, 1, 1]
    shape[2 - axis] = N  # array axes are (z,y,x)
    left = np.broadcast_to(left.reshape(shape), (N, N, N))
    rho = np.where(left, 1.0, 0.125).astype(dtype)
    P = np.where(left, 1.0, 0.1).astype(dtype)
    z = np.zeros((N, N, N), dtype)
    return prim_to_cons(rho, z, z, z, P, gamma)


# C2: spherical blast on an N^3 periodic grid, dh = 1, centre at the grid node (N/2,N/2,N/2);
# the cells with centre distance <= radius share total energy 1 (BASELINE.json configs[1]).
def blast_grid(N=128, radius=3.0, gamma=5.0 / 3.0, p_ambient=1e-5, dtype=np.float32):
    c = np.arange(N) + 0.5 - N / 2
    r2 = c[:, None, None] ** 2 + c[None, :, None] ** 2 + c[None, None, :] ** 2
    inside = r2 <= radius * radius
    U = np.zeros((5, N, N, N), dtype)
    U[0] = 1.0
    U[4] = p_ambient / (gamma - 1.0)
    U[4][inside] = 1.0 / inside.sum()
    return U


# C4: Kelvin-Helmholtz shear layer on an (Nz,Ny,Nx) periodic box, dh = 1/Ny-equivalent given by caller.
def kh_grid(shape=(64, 64, 64), gamma=1.4, amp=0.01, seed=0, dtype=np.float32):
    nz, ny, nx = shape
    rng = np.random.default_rng(seed)
    phi, psi = rng.uniform(0, 2 * np.pi, 4), rng.uniform(0, 2 * np.pi, 4)
    x = ((np.arange(nx) + 0.5) / nx)[None, None, :]
    y = ((np.arange(ny) + 0.5) / ny)[None, :, None]
    z = ((np.arange(nz) + 0.5) / nz)[:, None, None]
    band = np.broadcast_to(np.abs(y - 0.5) < 0.25, shape)
    rho = np.where(band, 2.0, 1.0)
    vx = np.where(band, 0.5, -0.5)
    vy = np.zeros(shape)
    for m in range(4):
        vy = vy + amp * np.sin(2 * np.pi * (m + 1) * x + phi[m]) * np.cos(2 * np.pi * z + psi[m]) / 2
    P = np.full(shape, 2.5)
    vz = np.zeros(shape)
    return prim_to_cons(rho.astype(dtype), vx.astype(dtype), vy.astype(dtype), vz.astype(dtype), P.astype(dtype), gamma)


# C5: random-phase "turbulent" velocity field, Mach ~ 1, |v_hat|^2 ~ k^-4 for 1 <= |k| <= kmax
def turbulence_grid(N=64, gamma=5.0 / 3.0, kmax=32, seed=0, dtype=np.float32):
    rng = np.random.default_rng(seed)
    k1 = np.fft.fftfreq(N, 1.0 / N)
    kr = np.fft.rfftfreq(N, 1.0 / N)
    k2 = k1[:, None, None] ** 2 + k1[None, :, None] ** 2 + kr[None, None, :] ** 2
    amp = np.where((k2 >= 1) & (k2 <= kmax * kmax), np.maximum(k2, 1.0) ** -1.0, 0.0)  # |v_hat| ~ k^-2
    v = []
    for _ in range(3):
        ph = rng.uniform(0, 2 * np.pi, amp.shape)
        v.append(np.fft.irfftn(amp * np.exp(1j * ph), s=(N, N, N), axes=(0, 1, 2)))
    v = np.stack(v)
    v *= 1.0 / np.sqrt((v ** 2).sum(0).mean())  # 3-D rms |v| = 1, c = 1  => Mach ~ 1
    rho = np.ones((N, N, N))
    P = np.full((N, N, N), 0.6)
    return prim_to_cons(rho.astype(dtype), v[0].astype(dtype), v[1].astype(dtype), v[2].astype(dtype),
                        P.astype(dtype), gamma)


# ------------------------------------------------------------------------------------------
# C3: AMR-shaped batch of independent padded groups (BASELINE.json configs[2]).
# Per group n and field q in (rho, P, vx, vy, vz): smooth unit-variance field
#   g_q(x) = sqrt(2/M) sum_{m<M} cos(2 pi k_m.x / S + phi_m),  k_m integer in {-2..2}^3 \ {0}
# rho = exp(0.5 g_rho), P = exp(0.3 g_P), v_d = 0.5 sqrt(gamma P / rho) g_d.
# Wave numbers and phases come from numpy Philox keyed by (seed, first group of the chunk);
# fields are evaluated with torch on `device` (CPU for tests, CUDA for the bench) in fp64.
def amr_batch(Ng, g=3, gamma=5.0 / 3.0, seed=0, dtype="float32", device="cpu", M=8, chunk=64):
    import torch

    S = PS + 2 * g
    tdt = {"float32": torch.float32, "float64": torch.float64}[str(dtype).replace("torch.", "")]
    out = torch.empty((Ng, 5, S, S, S), dtype=tdt, device=device)
    ax = torch.arange(S, dtype=torch.float64, device=device) * (2 * np.pi / S)
    for n0 in range(0, Ng, chunk):
        n1 = min(Ng, n0 + chunk)
        rng = np.random.Generator(np.random.Philox(key=[seed, n0]))
        k = rng.integers(-2, 3, size=(n1 - n0, 5, M, 3))
        zero = (k == 0).all(-1)
        k[zero] = (1, 0, 0)
        phi = rng.uniform(0, 2 * np.pi, size=(n1 - n0, 5, M))
        kt = torch.from_numpy(k).to(device=device, dtype=torch.float64)
        pt = torch.from_numpy(phi).to(device=device)
        f = torch.zeros((n1 - n0, 5, S, S, S), dtype=torch.float64, device=device)
        for m in range(M):
            arg = (kt[:, :, m, 2, None, None, None] * ax[None, None, :, None, None]
                   + kt[:, :, m, 1, None, None, None] * ax[None, None, None, :, None]
                   + kt[:, :, m, 0, None, None, None] * ax[None, None, None, None, :]
                   + pt[:, :, m, None, None, None])
            f += torch.cos(arg)
        f *= np.sqrt(2.0 / M)
        rho = torch.exp(0.5 * f[:, 0])
        P = torch.exp(0.3 * f[:, 1])
        cs = torch.sqrt(gamma * P / rho)
        vx, vy, vz = (0.5 * cs * f[:, 2 + d] for d in range(3))
        E = P / (gamma - 1.0) + 0.5 * rho * (vx * vx + vy * vy + vz * vz)
        out[n0:n1] = torch.stack([rho, rho * vx, rho * vy, rho * vz, E], 1).to(tdt)
    return out
