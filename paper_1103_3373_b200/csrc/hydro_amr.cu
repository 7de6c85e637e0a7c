// hydro_amr.cu -- the consumer of hydro_solve's `face_flux`: coarse-fine flux fix-up and fine -> coarse
// restriction after the fluid update of two adjacent AMR levels ("store the fluxes across the boundaries of all
// grid patches ... only necessary in AMR"; PAPER.md:137 the "coarse-grid correction", a CPU task in the paper).
// Reading S25 of DESIGN.md; layouts and index lists in include/hydro.h.  HBM-bound index plumbing: one CTA per coarse-fine
// face (64 coarse faces x 5 variables), one thread per restricted coarse cell.  Part of the CUDA product path.
#include <cuda_runtime.h>
#include <cstdint>

#include "../../include/hydro.h"

namespace hydro {

constexpr int APS = 16, AHP = 8;

__device__ __forceinline__ float add_rn(float a, float b) { return __fadd_rn(a, b); }
__device__ __forceinline__ double add_rn(double a, double b) { return __dadd_rn(a, b); }
__device__ __forceinline__ float mul_rn(float a, float b) { return __fmul_rn(a, b); }
__device__ __forceinline__ double mul_rn(double a, double b) { return __dmul_rn(a, b); }

// U <- U + sigma (dt_c/dh_c) (F_c - mean of the 2 x 2 fine fluxes); block = one face entry, thread = (variable, b, a)
template <class R>
__global__ void __launch_bounds__(320) fluxfix_kernel(R* __restrict__ coarse_out, const R* __restrict__ coarse_flux,
                                                      const R* __restrict__ fine_flux, const int* __restrict__ faces, R nu) {
  const int* f = faces + 7 * blockIdx.x;
  const int fine_group = f[0], d = f[1], fine_side = f[2], coarse_group = f[3];
  const int c0[3] = {f[4], f[5], f[6]};
  const int t = threadIdx.x, q = t >> 6, b = (t >> 3) & 7, a = t & 7;
  const int layer = c0[d];
  const int cf = fine_side == 0 ? layer + 1 : layer;  // the coarse face: upper face of the layer if the fine group lies above it
  const int s_c = cf >> 3;                            // 0, 8, 16 -> plane 0, 1, 2
  const R sigma = fine_side == 0 ? R(1) : R(-1);
  const int t1 = d == 0 ? 1 : 0, t2 = d == 2 ? 1 : 2;  // in-plane axes, lower axis fastest
  int c[3];
  c[d] = layer;
  c[t1] = c0[t1] + a;
  c[t2] = c0[t2] + b;
  const size_t plane_n = APS * APS, cell_n = (size_t)APS * APS * APS;
  const R fc = coarse_flux[(((size_t)coarse_group * 9 + (3 * d + s_c)) * 5 + q) * plane_n + (size_t)c[t2] * APS + c[t1]];
  const R* ff = fine_flux + (((size_t)fine_group * 9 + (3 * d + 2 * fine_side)) * 5 + q) * plane_n;
  const R fbar = mul_rn(add_rn(add_rn(ff[(2 * b) * APS + 2 * a], ff[(2 * b) * APS + 2 * a + 1]),
                               add_rn(ff[(2 * b + 1) * APS + 2 * a], ff[(2 * b + 1) * APS + 2 * a + 1])), R(0.25));
  // a coarse cell may touch refined patches across several of its faces: the contributions of different entries meet here
  atomicAdd(coarse_out + ((size_t)coarse_group * 5 + q) * cell_n + ((size_t)c[2] * APS + c[1]) * APS + c[0],
            mul_rn(mul_rn(sigma, nu), add_rn(fc, -fbar)));
}

// every fine group of the map replaces 8^3 coarse cells by the means of its 2 x 2 x 2 fine cells
template <class R>
__global__ void __launch_bounds__(256) restrict_kernel(const R* __restrict__ fine_out, R* __restrict__ coarse_out,
                                                       const int* __restrict__ map) {
  const int* m = map + 5 * blockIdx.y;
  const int idx = blockIdx.x * 256 + threadIdx.x;  // (q, k, j, i) over 5 x 8^3
  if (idx >= 5 * AHP * AHP * AHP) return;
  const int q = idx >> 9, k = (idx >> 6) & 7, j = (idx >> 3) & 7, i = idx & 7;
  const size_t cell_n = (size_t)APS * APS * APS;
  const R* F = fine_out + ((size_t)m[0] * 5 + q) * cell_n + ((size_t)(2 * k) * APS + 2 * j) * APS + 2 * i;
  const R lo = add_rn(add_rn(F[0], F[1]), add_rn(F[APS], F[APS + 1]));
  const R hi = add_rn(add_rn(F[APS * APS], F[APS * APS + 1]), add_rn(F[APS * APS + APS], F[APS * APS + APS + 1]));
  coarse_out[((size_t)m[1] * 5 + q) * cell_n + ((size_t)(m[4] + k) * APS + (m[3] + j)) * APS + (m[2] + i)] = mul_rn(add_rn(lo, hi), R(0.125));
}

template <class R> __global__ void flux_accum_kernel(R* __restrict__ acc, const R* __restrict__ ff, size_t n, R w) {
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x)
    acc[i] = add_rn(acc[i], mul_rn(w, ff[i]));
}

template <class R>
static int fluxfix_impl(R* coarse_out, const R* coarse_flux, const R* fine_flux, const int* faces, int nfaces, R dt_c, R dh_c, cudaStream_t st) {
  if (nfaces < 0) return HYDRO_E_COUNT;
  if (nfaces == 0) return HYDRO_OK;
  if (!coarse_out || !coarse_flux || !fine_flux || !faces) return HYDRO_E_NULL;
  if (((uintptr_t)coarse_out & 15) || ((uintptr_t)coarse_flux & 15) || ((uintptr_t)fine_flux & 15) || ((uintptr_t)faces & 3)) return HYDRO_E_ALIGN;
  if (!(dh_c > R(0)) || !(dt_c >= R(0))) return HYDRO_E_VALUE;
  fluxfix_kernel<R><<<nfaces, 320, 0, st>>>(coarse_out, coarse_flux, fine_flux, faces, dt_c / dh_c);
  return (int)cudaGetLastError();
}
template <class R> static int restrict_impl(const R* fine_out, R* coarse_out, const int* map, int n, cudaStream_t st) {
  if (n < 0) return HYDRO_E_COUNT;
  if (n == 0) return HYDRO_OK;
  if (!fine_out || !coarse_out || !map) return HYDRO_E_NULL;
  if (((uintptr_t)coarse_out & 15) || ((uintptr_t)fine_out & 15) || ((uintptr_t)map & 3)) return HYDRO_E_ALIGN;
  restrict_kernel<R><<<dim3(10, n), 256, 0, st>>>(fine_out, coarse_out, map);
  return (int)cudaGetLastError();
}
template <class R> static int accum_impl(R* acc, const R* ff, long long n, R w, cudaStream_t st) {
  if (n < 0) return HYDRO_E_COUNT;
  if (n == 0) return HYDRO_OK;
  if (!acc || !ff) return HYDRO_E_NULL;
  long long blocks = (n + 255) / 256;
  if (blocks > 148 * 16) blocks = 148 * 16;
  flux_accum_kernel<R><<<(unsigned)blocks, 256, 0, st>>>(acc, ff, (size_t)n, w);
  return (int)cudaGetLastError();
}

}  // namespace hydro

extern "C" {
int hydro_fluxfix_f32(float* coarse_out, const float* coarse_flux, const float* fine_flux, const int* faces, int nfaces, float dt_c,
                      float dh_c, hydro_stream_t stream) {
  return hydro::fluxfix_impl<float>(coarse_out, coarse_flux, fine_flux, faces, nfaces, dt_c, dh_c, (cudaStream_t)stream);
}
int hydro_fluxfix_f64(double* coarse_out, const double* coarse_flux, const double* fine_flux, const int* faces, int nfaces, double dt_c,
                      double dh_c, hydro_stream_t stream) {
  return hydro::fluxfix_impl<double>(coarse_out, coarse_flux, fine_flux, faces, nfaces, dt_c, dh_c, (cudaStream_t)stream);
}
int hydro_restrict_f32(const float* fine_out, float* coarse_out, const int* map, int n, hydro_stream_t stream) {
  return hydro::restrict_impl<float>(fine_out, coarse_out, map, n, (cudaStream_t)stream);
}
int hydro_restrict_f64(const double* fine_out, double* coarse_out, const int* map, int n, hydro_stream_t stream) {
  return hydro::restrict_impl<double>(fine_out, coarse_out, map, n, (cudaStream_t)stream);
}
int hydro_flux_accum_f32(float* acc, const float* face_flux, long long n, float w, hydro_stream_t stream) {
  return hydro::accum_impl<float>(acc, face_flux, n, w, (cudaStream_t)stream);
}
int hydro_flux_accum_f64(double* acc, const double* face_flux, long long n, double w, hydro_stream_t stream) {
  return hydro::accum_impl<double>(acc, face_flux, n, w, (cudaStream_t)stream);
}
}
