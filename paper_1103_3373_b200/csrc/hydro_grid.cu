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

// one CTA per (group, variable, z plane of the padded group); threads sweep the S x S plane, x fastest
template <class R>
__global__ void __launch_bounds__(GRID_NT) gather_kernel(const R* __restrict__ grid, R* __restrict__ groups, int Gx, int Gy, int Gz,
                                                          int g, int bc) {
  const int S = PS + 2 * g, Nx = Gx * PS, Ny = Gy * PS, Nz = Gz * PS;
  long long b = blockIdx.x;
  const int k = (int)(b % S); b /= S;
  const int v = (int)(b % 5); b /= 5;
  const int n = (int)b;
  const int gx = n % Gx, gy = (n / Gx) % Gy, gz = n / (Gx * Gy);
  int z = gz * PS - g + k;
  if (bc == 0) z = z < 0 ? z + Nz : (z >= Nz ? z - Nz : z);
  else z = z < 0 ? 0 : (z >= Nz ? Nz - 1 : z);
  const R* src = grid + ((size_t)v * Nz + z) * Ny * Nx;
  R* dst = groups + (((size_t)n * 5 + v) * S + k) * S * S;
  for (int idx = threadIdx.x; idx < S * S; idx += GRID_NT) {
    const int j = idx / S, i = idx - j * S;
    int y = gy * PS - g + j, x = gx * PS - g + i;
    if (bc == 0) {
      y = y < 0 ? y + Ny : (y >= Ny ? y - Ny : y);
      x = x < 0 ? x + Nx : (x >= Nx ? x - Nx : x);
    } else {
      y = y < 0 ? 0 : (y >= Ny ? Ny - 1 : y);
      x = x < 0 ? 0 : (x >= Nx ? Nx - 1 : x);
    }
    dst[idx] = __ldg(src + (size_t)y * Nx + x);
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
  const long long blocks = Ng * 5 * (PS + 2 * nghost);
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
