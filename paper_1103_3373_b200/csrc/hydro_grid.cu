// hydro_grid.cu -- device-side preparation and closing steps for uniform grids.
//
// In the paper these are CPU/OpenMP tasks -- "the preparation step ... stores the interior and ghost-cell data of
// the patch groups" and the closing step copies the results back -- and take up to three times the GPU time
// (PAPER.md:127).  On a uniform mesh they are pure index plumbing: gather copies every patch group with its ghost
// zones out of a [5][Nz][Ny][Nx] grid (periodic wrap or zero-gradient clamp at the domain boundary), scatter copies
// the updated 16^3 interiors back.  No arithmetic; results are bit-exact copies.  Both are HBM-bound:
// gather moves 5 (16^3 + S^3) elements per group (the re-read ghost cells mostly hit L2), scatter 10 * 16^3.
#include <cuda_runtime.h>
#include <cstdint>

#include "../../include/hydro.h"
#include "hydro_math.cuh"

namespace hydro {

constexpr int GRID_NT = 256;

// one CTA per (group, variable), GATHER_PL z planes of the padded group per pass: warp w fetches the rows j = w, w+8, ...
// of all those planes (lane = x, so a lane's source column is computed once; all loads of a pass are in flight
// together), the planes are staged in shared memory and leave as 16-byte pieces: GATHER_PL destination planes are
// GATHER_PL * S*S contiguous elements starting on a 16-byte boundary.
template <class R>
__global__ void __launch_bounds__(GRID_NT) gather_kernel(const R* __restrict__ grid, R* __restrict__ groups, int Gx, int Gy, int Gz,
                                                          int g, int bc) {
  constexpr int VEC = 16 / sizeof(R), NWARP = GRID_NT / 32, MAXR = (32 + NWARP - 1) / NWARP;  // rows per warp and plane
  constexpr int GATHER_PL = 4;  // planes per pass (8 measured slower: ragged last pass, fewer resident CTAs)
  __shared__ __align__(16) R tile[GATHER_PL * 32 * 32];
  const int S = PS + 2 * g, SS = S * S, Nx = Gx * PS, Ny = Gy * PS, Nz = Gz * PS;
  const int v = blockIdx.x % 5, n = blockIdx.x / 5;
  const int gx = n % Gx, gy = (n / Gx) % Gy, gz = n / (Gx * Gy);
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  auto fold = [bc](int c, int N) {  // periodic wrap or zero-gradient clamp (ghost width <= 8 < 16 <= N)
    return bc == 0 ? (c < 0 ? c + N : (c >= N ? c - N : c)) : (c < 0 ? 0 : (c >= N ? N - 1 : c));
  };
  const R* src = grid + (size_t)v * Nz * Ny * Nx + fold(gx * PS - g + lane, Nx);
  size_t yo[MAXR];  // source row offsets of this warp's rows
#pragma unroll
  for (int r = 0; r < MAXR; ++r) yo[r] = (size_t)fold(gy * PS - g + min(warp + r * NWARP, S - 1), Ny) * Nx;
  uint4* dst = reinterpret_cast<uint4*>(groups + ((size_t)n * 5 + v) * S * SS);
  for (int k0 = 0; k0 < S; k0 += GATHER_PL) {
    const int np = min(GATHER_PL, S - k0);
    R val[GATHER_PL][MAXR];
#pragma unroll
    for (int q = 0; q < GATHER_PL; ++q) {
      const R* sp = src + (size_t)fold(gz * PS - g + min(k0 + q, S - 1), Nz) * Ny * Nx;
#pragma unroll
      for (int r = 0; r < MAXR; ++r) val[q][r] = (lane < S) ? __ldg(sp + yo[r]) : R(0);
    }
    __syncthreads();  // the previous pass has left the tile
    if (lane < S) {
#pragma unroll
      for (int q = 0; q < GATHER_PL; ++q)
#pragma unroll
        for (int r = 0; r < MAXR; ++r) {
          const int j = warp + r * NWARP;
          if (j < S && q < np) tile[q * SS + j * S + lane] = val[q][r];
        }
    }
    __syncthreads();
    const uint4* t4 = reinterpret_cast<const uint4*>(tile);
    for (int q = threadIdx.x; q < np * SS / VEC; q += GRID_NT) dst[(size_t)k0 * (SS / VEC) + q] = t4[q];
  }
}

// one CTA per (group, variable, 4 z planes); a thread moves one 16-byte piece of a 16-cell row
template <class R>
__global__ void __launch_bounds__(GRID_NT) scatter_kernel(const R* __restrict__ out, R* __restrict__ grid, int Gx, int Gy, int Gz) {
  constexpr int VEC = 16 / sizeof(R);          // elements per 16-byte piece
  constexpr int PPR = PS / VEC;                // pieces per row
  constexpr int ROWS = GRID_NT / PPR;          // rows per CTA pass
  const int Nx = Gx * PS, Ny = Gy * PS, Nz = Gz * PS;
  long long b = blockIdx.x;
  const int v = (int)(b % 5); b /= 5;
  const int n = (int)b;
  const int gx = n % Gx, gy = (n / Gx) % Gy, gz = n / (Gx * Gy);
  const uint4* src = reinterpret_cast<const uint4*>(out + ((size_t)n * 5 + v) * PS * PS * PS);
  const int piece = threadIdx.x % PPR, row0 = threadIdx.x / PPR;
  for (int row = row0; row < PS * PS; row += ROWS) {  // row = k * 16 + j
    const int k = row >> 4, j = row & 15;
    R* d = grid + (((size_t)v * Nz + gz * PS + k) * Ny + gy * PS + j) * Nx + gx * PS;
    reinterpret_cast<uint4*>(d)[piece] = src[row * PPR + piece];
  }
}

template <class R>
static int gather_impl(const R* grid, R* groups, int nx, int ny, int nz, int nghost, int bc, cudaStream_t st) {
  if (nx < 0 || ny < 0 || nz < 0 || nx % PS || ny % PS || nz % PS) return HYDRO_E_VALUE;
  if (nghost < 0 || nghost > 8) return HYDRO_E_GHOST;
  if (bc < 0 || bc > 1) return HYDRO_E_ENUM;
  const long long Ng = (long long)(nx / PS) * (ny / PS) * (nz / PS);
  if (Ng == 0) return HYDRO_OK;
  if (!grid || !groups) return HYDRO_E_NULL;
  if (((uintptr_t)grid & 15) || ((uintptr_t)groups & 15)) return HYDRO_E_ALIGN;
  const long long blocks = Ng * 5;
  if (blocks > 0x7fffffffLL) return HYDRO_E_COUNT;
  gather_kernel<R><<<(unsigned)blocks, GRID_NT, 0, st>>>(grid, groups, nx / PS, ny / PS, nz / PS, nghost, bc);
  return (int)cudaGetLastError();
}

template <class R> static int scatter_impl(const R* out, R* grid, int nx, int ny, int nz, cudaStream_t st) {
  if (nx < 0 || ny < 0 || nz < 0 || nx % PS || ny % PS || nz % PS) return HYDRO_E_VALUE;
  const long long Ng = (long long)(nx / PS) * (ny / PS) * (nz / PS);
  if (Ng == 0) return HYDRO_OK;
  if (!grid || !out) return HYDRO_E_NULL;
  if (((uintptr_t)grid & 15) || ((uintptr_t)out & 15)) return HYDRO_E_ALIGN;
  if (Ng * 5 > 0x7fffffffLL) return HYDRO_E_COUNT;
  scatter_kernel<R><<<(unsigned)(Ng * 5), GRID_NT, 0, st>>>(out, grid, nx / PS, ny / PS, nz / PS);
  return (int)cudaGetLastError();
}

// entry points for hydro_advance (hydro_api.cu)
template <class R> int gather_impl_fwd(const R* grid, R* groups, int nx, int ny, int nz, int nghost, int bc, cudaStream_t st) {
  return gather_impl<R>(grid, groups, nx, ny, nz, nghost, bc, st);
}
template <class R> int scatter_impl_fwd(const R* out, R* grid, int nx, int ny, int nz, cudaStream_t st) {
  return scatter_impl<R>(out, grid, nx, ny, nz, st);
}
template int gather_impl_fwd<float>(const float*, float*, int, int, int, int, int, cudaStream_t);
template int gather_impl_fwd<double>(const double*, double*, int, int, int, int, int, cudaStream_t);
template int scatter_impl_fwd<float>(const float*, float*, int, int, int, cudaStream_t);
template int scatter_impl_fwd<double>(const double*, double*, int, int, int, cudaStream_t);

}  // namespace hydro

extern "C" {
int hydro_gather_f32(const float* grid, float* groups, int nx, int ny, int nz, int nghost, int bc, hydro_stream_t stream) {
  return hydro::gather_impl<float>(grid, groups, nx, ny, nz, nghost, bc, (cudaStream_t)stream);
}
int hydro_gather_f64(const double* grid, double* groups, int nx, int ny, int nz, int nghost, int bc, hydro_stream_t stream) {
  return hydro::gather_impl<double>(grid, groups, nx, ny, nz, nghost, bc, (cudaStream_t)stream);
}
int hydro_scatter_f32(const float* out, float* grid, int nx, int ny, int nz, hydro_stream_t stream) {
  return hydro::scatter_impl<float>(out, grid, nx, ny, nz, (cudaStream_t)stream);
}
int hydro_scatter_f64(const double* out, double* grid, int nx, int ny, int nz, hydro_stream_t stream) {
  return hydro::scatter_impl<double>(out, grid, nx, ny, nz, (cudaStream_t)stream);
}
}
