// hydro_lean_grid.cuh -- uniform-grid mode of the fused MHM and VL kernels (hydro_solve_grid_*: the ghost-zone
// preparation is folded into the solver): the raw planes of a patch group are fetched from the grid [5][Nz][Ny][Nx] itself
// with element-wise asynchronous copies, ghost cells folded at the domain boundary (periodic wrap or zero-gradient clamp),
// and the updated cells go straight back into the output grid.  The CTU kernel carries its own copy of this feed
// (hydro_lean_ctu.cuh), written before the other two kernels had a grid mode.
#pragma once
#include "hydro_launch.cuh"
#include "hydro_ptx.cuh"

namespace hydro {

// SWP: cells per row / rows per plane of a raw plane (16 + 2 GW); NPL: planes per group; NT: threads of the CTA
template <class R, int SWP, int NPL, int NT> struct GridFeed {
  int pl, m, gpk;  // plane within the group, group counter of this CTA, packed group coordinates (10 bits each)
  __device__ __forceinline__ void reset() { pl = 0; m = 0; gpk = 0; }
  static __device__ __forceinline__ int fold(int c, int N, int bc) {
    return bc == 0 ? (c < 0 ? c + N : (c >= N ? c - N : c)) : (c < 0 ? 0 : (c >= N ? N - 1 : c));
  }
  // every thread copies its share of the next raw plane of this CTA's group sequence into dst[5][SWP * SWP] and commits one
  // cp.async group (also when the sequence is exhausted: the wait_group arithmetic stays uniform)
  __device__ __forceinline__ void feed(const GridIO<R>& gio, int my_groups, R* dst, int tid) {
    constexpr int GW = (SWP - PS) / 2;
    if (m < my_groups) {
      const int Nx = gio.Gx * PS, Ny = gio.Gy * PS, Nz = gio.Gz * PS;
      const size_t N2 = (size_t)Ny * Nx, N3 = N2 * Nz;
      if (pl == 0) {
        const int grp = (int)blockIdx.x + m * (int)gridDim.x;
        gpk = (grp % gio.Gx) | (((grp / gio.Gx) % gio.Gy) << 10) | ((grp / (gio.Gx * gio.Gy)) << 20);
      }
      const int x0 = (gpk & 1023) * PS - GW, y0 = ((gpk >> 10) & 1023) * PS - GW, z0 = (gpk >> 20) * PS - GW;
      const R* zsrc = gio.gin + (size_t)fold(z0 + pl, Nz, gio.bc) * N2;
#pragma unroll
      for (int r = 0; r < (SWP * SWP + NT - 1) / NT; ++r) {
        const int pos = tid + r * NT;
        if (pos < SWP * SWP) {
          const int j = pos / SWP, i = pos - j * SWP;
          const R* sp = zsrc + (size_t)fold(y0 + j, Ny, gio.bc) * Nx + fold(x0 + i, Nx, gio.bc);
#pragma unroll
          for (int q = 0; q < 5; ++q) { cp_async_elem(dst + q * (SWP * SWP) + pos, sp); sp += N3; }
        }
      }
      if (++pl == NPL) { pl = 0; ++m; }
    }
    cp_async_commit();
  }
};

// index of interior cell (ci, cj, 0) of patch group grp in a grid [Nz][Ny][Nx]; a plane is N2 = Ny Nx cells further, a variable N3
template <class R> __device__ __forceinline__ size_t grid_cell0(const GridIO<R>& gio, size_t grp, int ci, int cj) {
  const int gi = (int)grp, gx = gi % gio.Gx, gy = (gi / gio.Gx) % gio.Gy, gz = gi / (gio.Gx * gio.Gy);
  const int Nx = gio.Gx * PS, Ny = gio.Gy * PS;
  return ((size_t)(gz * PS) * Ny + gy * PS + cj) * Nx + gx * PS + ci;
}

}  // namespace hydro
