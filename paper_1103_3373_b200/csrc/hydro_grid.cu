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
constexpr int GATHER_BRICK = 4;  // 8 measured the same; plain x-y-z order reads the z ghost zones from HBM twice

// One CTA per patch group.  A thread owns up to MAXE PAIRS of in-plane positions (j, i), (j, i + 1) of the padded group (S is
// even, so a pair never straddles a row) -- consecutive threads own consecutive destination pairs, so every store instruction
// of a warp is one contiguous 256- (512-) byte piece -- and forms their folded source offsets ONCE: they are the same for
// all S z planes and all five variables, so that the loop over the 5 S planes is nothing but loads and paired stores off a
// uniform plane base (GATHER_UN planes, 4 GATHER_UN loads per thread, in flight together).  The two sources of a pair are loaded separately (they are not
// adjacent where the ghost zone wraps around the domain).  Round 1's kernel (rows staged through shared memory) spent 27
// warp instructions per 22-element row on index arithmetic and predicates and was bound by instruction ISSUE (72 % of the
// issue slots busy at 3.1 TB/s); this one needs about 3.  CTAs walk the groups in bricks of 4 x 4 x 4, so that the ghost
// zones a group shares with its neighbours along z are still in L2 when the neighbour reads them (in plain x-y-z order they
// are one whole z layer of groups -- hundreds of MB of traffic -- apart and came from HBM twice).
template <class R> struct Pair;
template <> struct Pair<float> { using type = float2; };
template <> struct Pair<double> { using type = double2; };
template <class R>
__global__ void __launch_bounds__(GRID_NT) gather_kernel(const R* __restrict__ grid, R* __restrict__ groups, int Gx, int Gy, int Gz,
                                                          int g, int bc) {
  using P2 = typename Pair<R>::type;
  constexpr int MAXE = (32 * 32 / 2 + GRID_NT - 1) / GRID_NT;  // S <= 32
  constexpr int GATHER_UN = 2, BR = GATHER_BRICK;
  const int S = PS + 2 * g, SS = S * S, Nx = Gx * PS, Ny = Gy * PS, Nz = Gz * PS;
  // brick order: full bricks first (x fastest inside a brick), then the ragged remainder in plain order
  int gx, gy, gz;
  {
    const int bx = Gx / BR, by = Gy / BR, bz = Gz / BR, nfull = bx * by * bz * BR * BR * BR;
    int n = blockIdx.x;
    if (n < nfull) {
      const int in = n % (BR * BR * BR), b = n / (BR * BR * BR);
      gx = (b % bx) * BR + in % BR; gy = ((b / bx) % by) * BR + (in / BR) % BR; gz = (b / (bx * by)) * BR + in / (BR * BR);
    } else {  // groups outside the full bricks, enumerated in x-y-z order
      n -= nfull;
      const int fx = bx * BR, fy = by * BR, fz = bz * BR;
      gx = gy = gz = 0;
      for (int z = 0, c = 0; z < Gz; ++z)
        for (int y = 0; y < Gy; ++y) {
          const int skip = (z < fz && y < fy) ? fx : 0, cnt = Gx - skip;
          if (n < c + cnt) { gx = skip + (n - c); gy = y; gz = z; z = Gz; break; }
          c += cnt;
        }
    }
  }
  const int n = (gz * Gy + gy) * Gx + gx;
  auto fold = [bc](int c, int N) {  // periodic wrap or zero-gradient clamp (ghost width <= 8 < 16 <= N)
    return bc == 0 ? (c < 0 ? c + N : (c >= N ? c - N : c)) : (c < 0 ? 0 : (c >= N ? N - 1 : c));
  };
  int s0[MAXE], s1[MAXE];  // source offsets within a z plane of the grid of the pair's two elements; s0 = -1: no pair
#pragma unroll
  for (int r = 0; r < MAXE; ++r) {
    const int idx = 2 * ((int)threadIdx.x + r * GRID_NT);
    const int j = idx / S, i = idx - j * S;
    const int row = fold(gy * PS - g + j, Ny) * Nx;
    s0[r] = idx < SS ? row + fold(gx * PS - g + i, Nx) : -1;
    s1[r] = row + fold(gx * PS - g + i + 1, Nx);
  }
  // byte offsets of the S source planes within a variable (folded along z), formed once per CTA
  __shared__ long long zoff[32];
  const size_t N2 = (size_t)Ny * Nx;
  if (threadIdx.x < S) zoff[threadIdx.x] = (long long)((size_t)fold(gz * PS - g + (int)threadIdx.x, Nz) * N2 * sizeof(R));
  __syncthreads();
  P2* dst = reinterpret_cast<P2*>(groups + (size_t)n * 5 * S * SS) + threadIdx.x;
  const char* vp = reinterpret_cast<const char*>(grid);
  const size_t vstride = (size_t)Nz * N2 * sizeof(R);
  const int half = SS / 2;
  for (int v = 0; v < 5; ++v) {
    for (int k0 = 0; k0 < S; k0 += GATHER_UN) {  // S is even: GATHER_UN = 2 leaves no remainder
      P2 val[GATHER_UN][MAXE];
#pragma unroll
      for (int u = 0; u < GATHER_UN; ++u) {
        const R* sp = reinterpret_cast<const R*>(vp + zoff[k0 + u]);
        asm volatile("" : "+l"(sp));  // a finished plane base: every load address is then ONE wide multiply-add off it
#pragma unroll
        for (int r = 0; r < MAXE; ++r)
          if (s0[r] >= 0) { val[u][r].x = __ldg(sp + s0[r]); val[u][r].y = __ldg(sp + s1[r]); }
      }
#pragma unroll
      for (int u = 0; u < GATHER_UN; ++u) {
#pragma unroll
        for (int r = 0; r < MAXE; ++r)
          if (s0[r] >= 0) dst[u * half + r * GRID_NT] = val[u][r];
      }
      dst += GATHER_UN * half;
    }
    vp += vstride;
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
  const long long blocks = Ng;
  if (blocks * 5 > 0x7fffffffLL || (long long)nx * ny > 0x7fffffffLL) return HYDRO_E_COUNT;
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
