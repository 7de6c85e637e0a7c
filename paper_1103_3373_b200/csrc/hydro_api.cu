// hydro_api.cu -- the C ABI of include/hydro.h: argument validation, variant dispatch, the
// hydro_dt reduction kernel and the host-buffer streaming pipeline.
#include <cuda_runtime.h>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <new>
#include <vector>

#include "../../include/hydro.h"
#include "hydro_launch.cuh"

namespace hydro {

// gather / scatter of hydro_grid.cu, for hydro_advance
template <class R> int gather_impl_fwd(const R* grid, R* groups, int nx, int ny, int nz, int nghost, int bc, cudaStream_t st);
template <class R> int scatter_impl_fwd(const R* out, R* grid, int nx, int ny, int nz, cudaStream_t st);

// ---- dispatch tables ---------------------------------------------------------------------------
#define DECL_STAGED(R, S, RC, RS) extern template cudaError_t launch_staged<R, S, RC, RS>(const SolveArgs<R>&);
#define DECL_LEAN(R, S, RC, RS) extern template cudaError_t launch_lean<R, S, RC, RS>(const SolveArgs<R>&);
#define FOR_RS(M, R, S, RC) M(R, S, RC, RS_EXACT) M(R, S, RC, RS_HLLE) M(R, S, RC, RS_HLLC) M(R, S, RC, RS_ROE)
#define FOR_RC(M, R, S) FOR_RS(M, R, S, RECON_PLM) FOR_RS(M, R, S, RECON_PPM)
#define FOR_S(M, R) FOR_RC(M, R, SCHEME_MHM) FOR_RC(M, R, SCHEME_VL) FOR_RC(M, R, SCHEME_CTU)
FOR_S(DECL_STAGED, float)
FOR_S(DECL_STAGED, double)
FOR_S(DECL_LEAN, float)
FOR_S(DECL_LEAN, double)

template <class R> static LaunchFn<R> staged_fn(int scheme, int recon, int rs) {
#define ROW(R_, S, RC) {&launch_staged<R_, S, RC, RS_EXACT>, &launch_staged<R_, S, RC, RS_HLLE>, \
                        &launch_staged<R_, S, RC, RS_HLLC>, &launch_staged<R_, S, RC, RS_ROE>}
  static const LaunchFn<R> t[3][2][4] = {
      {ROW(R, SCHEME_MHM, RECON_PLM), ROW(R, SCHEME_MHM, RECON_PPM)},
      {ROW(R, SCHEME_VL, RECON_PLM), ROW(R, SCHEME_VL, RECON_PPM)},
      {ROW(R, SCHEME_CTU, RECON_PLM), ROW(R, SCHEME_CTU, RECON_PPM)}};
#undef ROW
  return t[scheme][recon][rs];
}
template <class R> static LaunchFn<R> lean_fn(int scheme, int recon, int rs) {
#define ROW(R_, S, RC) {&launch_lean<R_, S, RC, RS_EXACT>, &launch_lean<R_, S, RC, RS_HLLE>, \
                        &launch_lean<R_, S, RC, RS_HLLC>, &launch_lean<R_, S, RC, RS_ROE>}
  static const LaunchFn<R> t[3][2][4] = {
      {ROW(R, SCHEME_MHM, RECON_PLM), ROW(R, SCHEME_MHM, RECON_PPM)},
      {ROW(R, SCHEME_VL, RECON_PLM), ROW(R, SCHEME_VL, RECON_PPM)},
      {ROW(R, SCHEME_CTU, RECON_PLM), ROW(R, SCHEME_CTU, RECON_PPM)}};
#undef ROW
  return t[scheme][recon][rs];
}

// ---- hydro_dt (DESIGN.md c6) -------------------------------------------------------
// Non-negative IEEE values order like their bit patterns, and the canonical NaN pattern is larger
// than +inf, so one integer atomicMax per CTA yields "max, or NaN if any cell was bad".
constexpr int DT_NT = 256;

template <class R> struct Vec2;
template <> struct Vec2<float> { using T = float2; };
template <> struct Vec2<double> { using T = double2; };

// wave speed of one cell, as bits: max-ordered, NaN pattern for a non-positive state (see above)
template <class R> __device__ __forceinline__ typename Bits<R>::U dt_cell(R rho, R mx, R my, R mz, R E, R gamma, int norm) {
  const R ir = m_rcp(rho);
  const R vx = mx * ir, vy = my * ir, vz = mz * ir;
  const R P = (gamma - R(1)) * (E - R(0.5) * rho * ((vx * vx + vy * vy) + vz * vz));
  const R c = m_sqrt(gamma * P * ir);
  const R ax = m_abs(vx), ay = m_abs(vy), az = m_abs(vz);
  const R s = norm == 0 ? m_max(m_max(ax, ay), az) + c : ((ax + ay) + az) + R(3) * c;
  const bool bad = !(rho > R(0)) || !(P > R(0)) || !(s == s);
  return bad ? Bits<R>::nan() : Bits<R>::of(s);
}

// A warp takes one "span": the 16 interior rows j of one z plane of one group, which are 16 S CONSECUTIVE elements per variable
// (the ghost columns between them included), and reads them as two-element vectors -- every load instruction of the warp
// is one contiguous 256 / 512-byte piece.  Ghost columns are masked after the load.  The interior rows of a plane share
// their 32-byte sectors with the ghost columns, so what HBM must deliver per interior cell is (16 + 2 g) / 16 of the
// algorithmic 5 sizeof(R) bytes: the ceiling of this kernel by algorithmic bytes is 16 / (16 + 2 g) of the copy peak (73 % at g = 3).
template <class R>
__global__ void __launch_bounds__(DT_NT) dt_kernel(const R* __restrict__ u, long long nspans, int g, R gamma, int norm,
                                                   typename Bits<R>::U* __restrict__ result) {
  using U = typename Bits<R>::U;
  using V = typename Vec2<R>::T;
  const int S = PS + 2 * g;
  const size_t nS = (size_t)S * S * S;
  const int lane = threadIdx.x & 31;
  const long long warp = ((long long)blockIdx.x * DT_NT + threadIdx.x) >> 5, nwarps = ((long long)gridDim.x * DT_NT) >> 5;
  const int npieces = PS * S / 2;  // two-element pieces per span
  U best = 0;
  for (long long sp = warp; sp < nspans; sp += nwarps) {
    const long long grp = sp >> 4;
    const int k = (int)(sp & 15);
    const V* b = reinterpret_cast<const V*>(u + (size_t)grp * 5 * nS + ((size_t)(k + g) * S + g) * S);
    for (int p0 = 0; p0 < npieces; p0 += 32 * 4) {
      V v[4][5];
#pragma unroll
      for (int t = 0; t < 4; ++t) {
        const int pc = p0 + t * 32 + lane;
#pragma unroll
        for (int q = 0; q < 5; ++q) {
          if (pc < npieces) v[t][q] = __ldg(b + q * (nS / 2) + pc);
          else { v[t][q].x = R(1); v[t][q].y = R(1); }
        }
      }
#pragma unroll
      for (int t = 0; t < 4; ++t) {
        const int pc = p0 + t * 32 + lane;
        if (pc < npieces) {
          const int e = 2 * pc, i0 = e % S;  // column of the first element of the piece within its row (S is even: same row)
          if (i0 >= g && i0 < g + PS) {
            const U bits = dt_cell<R>(v[t][0].x, v[t][1].x, v[t][2].x, v[t][3].x, v[t][4].x, gamma, norm);
            best = bits > best ? bits : best;
          }
          if (i0 + 1 >= g && i0 + 1 < g + PS) {
            const U bits = dt_cell<R>(v[t][0].y, v[t][1].y, v[t][2].y, v[t][3].y, v[t][4].y, gamma, norm);
            best = bits > best ? bits : best;
          }
        }
      }
    }
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    const U other = __shfl_xor_sync(0xffffffffu, best, o);
    best = other > best ? other : best;
  }
  __shared__ U wmax[DT_NT / 32];
  if ((threadIdx.x & 31) == 0) wmax[threadIdx.x >> 5] = best;
  __syncthreads();
  if (threadIdx.x == 0) {
    U m = wmax[0];
#pragma unroll
    for (int w = 1; w < DT_NT / 32; ++w) m = wmax[w] > m ? wmax[w] : m;
    atomicMax(result, m);
  }
}

static int g_sm_count = 0;
static int sm_count() {
  if (!g_sm_count) {
    int dev = 0, n = 0;
    if (cudaGetDevice(&dev) == cudaSuccess && cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && n > 0)
      g_sm_count = n;
    else
      g_sm_count = 148;
  }
  return g_sm_count;
}

template <class R>
static int dt_impl(const R* u, int Ng, int nghost, R gamma, int norm, R* max_speed, cudaStream_t st, bool accumulate = false) {
  if (Ng < 0) return HYDRO_E_COUNT;
  if (!max_speed || (Ng > 0 && !u)) return HYDRO_E_NULL;
  if (norm < 0 || norm > 1) return HYDRO_E_ENUM;
  if (nghost < 0 || nghost > 8) return HYDRO_E_GHOST;
  if (!(gamma > R(1))) return HYDRO_E_VALUE;
  if (((uintptr_t)u & 15) || ((uintptr_t)max_speed & (sizeof(R) - 1))) return HYDRO_E_ALIGN;
  if (!accumulate) {
    cudaError_t e = cudaMemsetAsync(max_speed, 0, sizeof(R), st);
    if (e != cudaSuccess) return (int)e;
  }
  if (Ng == 0) return HYDRO_OK;
  const long long nspans = (long long)Ng * PS;  // one per (group, interior z plane)
  long long blocks = (nspans * 32 + DT_NT - 1) / DT_NT;
  const long long cap = (long long)sm_count() * 8;
  if (blocks > cap) blocks = cap;
  dt_kernel<R><<<(unsigned)blocks, DT_NT, 0, st>>>(u, nspans, nghost, gamma, norm,
                                                  reinterpret_cast<typename Bits<R>::U*>(max_speed));
  return (int)cudaGetLastError();
}

// ---- hydro_solve ---------------------------------------------------------------------------------
struct Plan {
  int recon, g, impl;  // impl resolved to STAGED or FUSED
};

template <class R>
static int make_plan(const void* in, const void* out, const void* ff, int Ng, R dt, R dh, R gamma, int scheme, int riemann,
                     int limiter, const hydro_opts* o, bool device_ptrs, Par<R>& par, Plan& pl) {
  if (scheme < 0 || scheme > 2 || riemann < 0 || riemann > 3 || limiter < 0 || limiter > 3) return HYDRO_E_ENUM;
  const int recon = o ? o->recon : 0;
  const int fb = (o && o->roe_fallback) ? o->roe_fallback : 1;
  const int impl = o ? o->impl : 0;
  if (recon < 0 || recon > 1 || fb < 1 || fb > 3 || impl < 0 || impl > 2) return HYDRO_E_ENUM;
  if (o && (o->char_limit < 0 || o->char_limit > 1)) return HYDRO_E_ENUM;
  if (Ng < 0) return HYDRO_E_COUNT;
  if (Ng > 0 && (!in || !out)) return HYDRO_E_NULL;
  if (device_ptrs && (((uintptr_t)in & 15) || ((uintptr_t)out & 15) || ((uintptr_t)ff & 15))) return HYDRO_E_ALIGN;
  if (device_ptrs && o && o->status && ((uintptr_t)o->status & 7)) return HYDRO_E_ALIGN;
  const int gmin = min_ghost(scheme, recon);
  const int g = (o && o->nghost) ? o->nghost : gmin;
  if (g < gmin || g > 8) return HYDRO_E_GHOST;
  const double theta = (o && o->minmod_coeff != 0.0f) ? (double)o->minmod_coeff : 1.5;
  const bool device_dt = o && o->max_speed;  // then the `dt` argument is ignored (hydro.h): do not validate it
  if (!(gamma > R(1)) || !(dh > R(0)) || (!device_dt && !(dt >= R(0))) || !(theta >= 1.0 && theta <= 2.0)) return HYDRO_E_VALUE;
  if (o && (!(o->min_dens >= 0.0) || !(o->min_pres >= 0.0))) return HYDRO_E_VALUE;
  if (o && o->max_speed && (!(o->cfl > 0.0) || ((uintptr_t)o->max_speed & (sizeof(R) - 1)))) return HYDRO_E_VALUE;
  if (o && o->next_max_speed && (((uintptr_t)o->next_max_speed & (sizeof(R) - 1)) || o->next_max_speed == o->max_speed)) return HYDRO_E_ALIGN;
  if (o && (o->next_norm < 0 || o->next_norm > 1)) return HYDRO_E_ENUM;
  par.gamma = gamma;
  par.gm1 = gamma - R(1);
  par.igm1 = R(1) / par.gm1;
  par.ig1 = R(1) / (gamma + R(1));
  par.ig2 = R(0.5) / gamma;
  par.sA0 = (R)std::sqrt(2.0 / ((double)gamma + 1.0));
  par.nu = device_dt ? R(0) : dt / dh;
  par.hnu = R(0.5) * par.nu;
  par.theta = (R)theta;
  par.min_dens = o ? (R)o->min_dens : R(0);
  par.min_pres = o ? (R)o->min_pres : R(0);
  par.limiter = limiter;
  par.char_limit = o ? o->char_limit : 0;
  par.roe_fallback = fb;
  par.next_speed = (o && device_ptrs) ? static_cast<R*>(o->next_max_speed) : nullptr;
  par.next_norm = o ? o->next_norm : 0;
  const bool has = lean_fits((int)sizeof(R), scheme, recon, g);  // kernel exists and its tiles fit in shared memory
  if (impl == HYDRO_IMPL_FUSED && !has) return HYDRO_E_NOFUSED;
  pl.recon = recon;
  pl.g = g;
  pl.impl = (impl != HYDRO_IMPL_STAGED && has) ? HYDRO_IMPL_FUSED : HYDRO_IMPL_STAGED;
  return HYDRO_OK;
}

template <class R>
static int solve_impl(const R* in, R* out, R* ff, int Ng, R dt, R dh, R gamma, int scheme, int riemann, int limiter,
                      const hydro_opts* o, cudaStream_t st) {
  SolveArgs<R> a;
  Plan pl;
  const int rc = make_plan<R>(in, out, ff, Ng, dt, dh, gamma, scheme, riemann, limiter, o, true, a.par, pl);
  if (rc != HYDRO_OK) return rc;
  if (Ng == 0) {  // no-op, but the reduction of an empty update is defined: 0, as hydro_dt of no groups
    if (a.par.next_speed) return (int)cudaMemsetAsync(a.par.next_speed, 0, sizeof(R), st);
    return HYDRO_OK;
  }
  a.in = in;
  a.out = out;
  a.face_flux = ff;
  a.Ng = Ng;
  a.g = pl.g;
  a.max_speed = o ? static_cast<const R*>(o->max_speed) : nullptr;
  a.cfl = o ? (R)o->cfl : R(0);
  a.status = o ? o->status : nullptr;
  a.workspace = o ? o->workspace : nullptr;
  a.workspace_bytes = o ? o->workspace_bytes : 0;
  a.stream = st;
  a.grid = GridIO<R>{nullptr, nullptr, 0, 0, 0, 0};
  if (a.par.next_speed) {
    const cudaError_t e = cudaMemsetAsync(a.par.next_speed, 0, sizeof(R), st);
    if (e != cudaSuccess) return (int)e;
  }
  if (pl.impl == HYDRO_IMPL_STAGED) {
    if (!a.workspace || ((uintptr_t)a.workspace & 15) || a.workspace_bytes < staged_slot_bytes(scheme, pl.recon, sizeof(R)))
      return HYDRO_E_WORKSPACE;
    R* next = a.par.next_speed;
    a.par.next_speed = nullptr;  // the staged kernel has no fused reduction: hydro_dt on `out` after it
    const int rc2 = (int)staged_fn<R>(scheme, pl.recon, riemann)(a);
    if (rc2 != 0 || !next) return rc2;
    return dt_impl<R>(out, Ng, 0, gamma, a.par.next_norm, next, st, true);
  }
  return (int)lean_fn<R>(scheme, pl.recon, riemann)(a);
}

// variants hydro_solve_grid_* covers (one launch per step, ghost zones folded out of the grid by the fused kernels): every
// scheme, reconstruction, solver and limiter option; the one exception is VL with positivity floors, whose half step re-reads
// U^n of ghost cells from the batch (hydro_lean_vl.cuh S2) -- that combination takes the group path
static bool grid_mode_ok(int scheme, int limiter, const hydro_opts* o) {
  (void)limiter;
  const bool floors = o && (o->min_dens > 0.0 || o->min_pres > 0.0);
  return !(scheme == SCHEME_VL && floors);
}

// One update of a uniform grid in ONE launch: the fused kernel fetches its planes from grid_in (ghost zones folded
// at the domain boundary) and writes the updated cells into grid_out; no gather / scatter pass, no group buffers.
template <class R>
static int solve_grid_impl(const R* gin, R* gout, int nx, int ny, int nz, int bc, R dt, R dh, R gamma, int scheme, int riemann,
                           int limiter, const hydro_opts* o, cudaStream_t st) {
  if (nx < 0 || ny < 0 || nz < 0 || nx % PS || ny % PS || nz % PS) return HYDRO_E_VALUE;
  if (bc < 0 || bc > 1) return HYDRO_E_ENUM;
  const long long Ng = (long long)(nx / PS) * (ny / PS) * (nz / PS);
  if (Ng > 0x7fffffffLL / 64 || nx / PS > 1023 || ny / PS > 1023 || nz / PS > 1023) return HYDRO_E_COUNT;
  if (gin == gout && Ng > 0) return HYDRO_E_ALIGN;
  SolveArgs<R> a;
  Plan pl;
  hydro_opts oo;
  if (o) oo = *o; else std::memset(&oo, 0, sizeof(oo));
  oo.nghost = 0;  // ghost zones come from the grid: always the minimum width
  oo.impl = HYDRO_IMPL_FUSED;
  const int rc = make_plan<R>(gin, gout, nullptr, (int)Ng, dt, dh, gamma, scheme, riemann, limiter, &oo, true, a.par, pl);
  if (rc != HYDRO_OK) return rc;
  if (!grid_mode_ok(scheme, limiter, &oo)) return HYDRO_E_NOFUSED;  // callers fall back to gather -> hydro_solve -> scatter
  if (Ng == 0) return HYDRO_OK;
  a.in = nullptr;
  a.out = nullptr;
  a.face_flux = nullptr;
  a.Ng = (int)Ng;
  a.g = pl.g;
  a.max_speed = static_cast<const R*>(oo.max_speed);
  a.cfl = (R)oo.cfl;
  a.status = oo.status;
  a.workspace = nullptr;
  a.workspace_bytes = 0;
  a.stream = st;
  a.grid = GridIO<R>{gin, gout, nx / PS, ny / PS, nz / PS, bc};
  if (a.par.next_speed) {
    const cudaError_t e = cudaMemsetAsync(a.par.next_speed, 0, sizeof(R), st);
    if (e != cudaSuccess) return (int)e;
  }
  return (int)lean_fn<R>(scheme, pl.recon, riemann)(a);
}


// ---- hydro_advance: the multi-step driver of a uniform grid, entirely on the device ----------------
// elapsed time: t += cfl dh / max_speed in fp64, by one thread on the stream (the solver kernels take dt/dh = cfl / max_speed
// from the same scalar, hydro_opts::max_speed)
template <class R> __global__ void advance_time_kernel(double* t, const R* max_speed, double cfl_dh) { *t += cfl_dh / (double)*max_speed; }

constexpr size_t ADV_HEAD = 256;  // workspace head: two speed scalars (ping-pong) at offsets 0 and 64
template <class R> static size_t advance_bytes(int nx, int ny, int nz, int scheme, int limiter, const hydro_opts* o) {
  const size_t cells = (size_t)nx * ny * nz, Ng = cells / (PS * PS * PS);
  if (grid_mode_ok(scheme, limiter, o) && !(o && o->nghost)) return ADV_HEAD + 5 * cells * sizeof(R);  // the second grid
  const int recon = o ? o->recon : 0;
  const int g = (o && o->nghost) ? o->nghost : min_ghost(scheme, recon);
  const size_t S = PS + 2 * g;
  size_t b = ADV_HEAD + Ng * 5 * (S * S * S + (size_t)PS * PS * PS) * sizeof(R);  // padded groups + updated interiors
  b = (b + 255) & ~(size_t)255;
  if (!lean_fits((int)sizeof(R), scheme, recon, g) || (o && o->impl == HYDRO_IMPL_STAGED))
    b += hydro_staged_workspace_bytes((int)(Ng < 0x7fffffff ? Ng : 0x7fffffff), (int)sizeof(R), scheme, recon);
  return b;
}

template <class R>
static int advance_impl(R* grid, int nx, int ny, int nz, int bc, int steps, R dh, R gamma, int scheme, int riemann, int limiter,
                        const hydro_opts* o, void* work, size_t work_bytes, double* t_accum, cudaStream_t st) {
  if (steps < 0) return HYDRO_E_COUNT;
  if (nx < 0 || ny < 0 || nz < 0 || nx % PS || ny % PS || nz % PS) return HYDRO_E_VALUE;
  if (bc < 0 || bc > 1) return HYDRO_E_ENUM;
  if (scheme < 0 || scheme > 2 || riemann < 0 || riemann > 3 || limiter < 0 || limiter > 3) return HYDRO_E_ENUM;
  if (!o || !(o->cfl > 0.0)) return HYDRO_E_VALUE;
  if (o->recon < 0 || o->recon > 1) return HYDRO_E_ENUM;
  const size_t cells = (size_t)nx * ny * nz;
  if (steps == 0 || cells == 0) return HYDRO_OK;
  if (!grid || !work) return HYDRO_E_NULL;
  if (((uintptr_t)grid & 15) || ((uintptr_t)work & 255) || (t_accum && ((uintptr_t)t_accum & 7))) return HYDRO_E_ALIGN;
  if (work_bytes < advance_bytes<R>(nx, ny, nz, scheme, limiter, o)) return HYDRO_E_WORKSPACE;
  const long long Ngl = (long long)(cells / (PS * PS * PS));
  if (Ngl > 0x7fffffffLL / 64) return HYDRO_E_COUNT;
  const int Ng = (int)Ngl;
  unsigned char* w = static_cast<unsigned char*>(work);
  R* sp[2] = {reinterpret_cast<R*>(w), reinterpret_cast<R*>(w + 64)};
  hydro_opts oo = *o;
  oo.max_speed = nullptr;
  oo.next_max_speed = nullptr;
  const double cfl_dh = o->cfl * (double)dh;
  int rc;
  if (grid_mode_ok(scheme, limiter, o) && !o->nghost) {  // an explicit ghost width asks for the group path
    R* other = reinterpret_cast<R*>(w + ADV_HEAD);
    R* buf[2] = {grid, other};
    // wave speed of the start state: the interiors only (a gather with ghost width 0 into the second grid, used as scratch)
    rc = gather_impl_fwd<R>(grid, other, nx, ny, nz, 0, bc, st);
    if (rc != HYDRO_OK) return rc;
    rc = dt_impl<R>(other, Ng, 0, gamma, 0, sp[0], st);
    if (rc != HYDRO_OK) return rc;
    for (int k = 0; k < steps; ++k) {
      oo.max_speed = sp[k & 1];
      oo.next_max_speed = sp[(k + 1) & 1];
      if (t_accum) advance_time_kernel<R><<<1, 1, 0, st>>>(t_accum, sp[k & 1], cfl_dh);
      rc = solve_grid_impl<R>(buf[k & 1], buf[(k + 1) & 1], nx, ny, nz, bc, R(0), dh, gamma, scheme, riemann, limiter, &oo, st);
      if (rc != HYDRO_OK) return rc;
    }
    if (steps & 1) {  // the result sits in the scratch grid: hand it back in the caller's
      const cudaError_t e = cudaMemcpyAsync(grid, other, 5 * cells * sizeof(R), cudaMemcpyDeviceToDevice, st);
      if (e != cudaSuccess) return (int)e;
    }
    return HYDRO_OK;
  }
  const int recon = o->recon;
  const int g = o->nghost ? o->nghost : min_ghost(scheme, recon);
  if (g < min_ghost(scheme, recon) || g > 8) return HYDRO_E_GHOST;
  const size_t S = PS + 2 * g;
  R* groups = reinterpret_cast<R*>(w + ADV_HEAD);
  R* out = groups + (size_t)Ng * 5 * S * S * S;
  size_t used = ADV_HEAD + (size_t)Ng * 5 * (S * S * S + (size_t)PS * PS * PS) * sizeof(R);
  used = (used + 255) & ~(size_t)255;
  oo.nghost = g;
  oo.workspace = w + used;
  oo.workspace_bytes = work_bytes - used;
  for (int k = 0; k < steps; ++k) {
    rc = gather_impl_fwd<R>(grid, groups, nx, ny, nz, g, bc, st);
    if (rc != HYDRO_OK) return rc;
    if (k == 0) {
      rc = dt_impl<R>(groups, Ng, g, gamma, 0, sp[0], st);
      if (rc != HYDRO_OK) return rc;
    }
    oo.max_speed = sp[k & 1];
    oo.next_max_speed = sp[(k + 1) & 1];
    if (t_accum) advance_time_kernel<R><<<1, 1, 0, st>>>(t_accum, sp[k & 1], cfl_dh);
    rc = solve_impl<R>(groups, out, nullptr, Ng, R(0), dh, gamma, scheme, riemann, limiter, &oo, st);
    if (rc != HYDRO_OK) return rc;
    rc = scatter_impl_fwd<R>(out, grid, nx, ny, nz, st);
    if (rc != HYDRO_OK) return rc;
  }
  return HYDRO_OK;
}

}  // namespace hydro

// ---- the host-buffer streaming pipeline ---------------------------------------
struct hydro_pipeline {
  int prec, g, chunk, ns;
  size_t in_elems, out_elems, ff_elems;  // per group
  std::vector<cudaStream_t> streams;
  std::vector<void*> d_in, d_out, d_ff, d_ws;
  size_t ws_bytes;
  long long* d_status;
  void* d_speed;  // [ns] per-stream running maxima of the updated state's wave speed
};

namespace hydro {
template <class R>
static int pipeline_solve(hydro_pipeline* p, const R* in, R* out, R* ff, int Ng, R dt, R dh, R gamma, int scheme, int riemann,
                          int limiter, const hydro_opts* o, long long* status_host, R* max_speed_host) {
  if (!p) return HYDRO_E_NULL;
  if (p->prec != (int)sizeof(R)) return HYDRO_E_VALUE;
  hydro_opts oo;
  if (o) oo = *o; else std::memset(&oo, 0, sizeof(oo));
  oo.nghost = p->g;
  oo.status = status_host ? p->d_status : nullptr;
  oo.max_speed = nullptr;
  oo.next_max_speed = nullptr;
  Par<R> par;
  Plan pl;
  int rc = make_plan<R>(in, out, ff, Ng, dt, dh, gamma, scheme, riemann, limiter, &oo, false, par, pl);
  if (rc != HYDRO_OK) return rc;
  if (Ng == 0) return HYDRO_OK;
  if (pl.impl == HYDRO_IMPL_STAGED) {
    const size_t need = hydro_staged_workspace_bytes(p->chunk, p->prec, scheme, pl.recon);
    if (p->ws_bytes < need) {  // (re)allocate per-stream scratch once for this variant
      p->ws_bytes = 0;  // nothing usable until every stream has its new scratch
      for (auto& w : p->d_ws) { if (w) cudaFree(w); w = nullptr; }
      for (auto& w : p->d_ws) if (cudaMalloc(&w, need) != cudaSuccess) return (int)cudaErrorMemoryAllocation;
      p->ws_bytes = need;
    }
  }
  if (status_host) cudaMemsetAsync(p->d_status, 0, 3 * sizeof(long long), p->streams[0]);
  if (max_speed_host) cudaMemsetAsync(p->d_speed, 0, p->ns * sizeof(double), p->streams[0]);
  if (status_host || max_speed_host) cudaStreamSynchronize(p->streams[0]);
  // on any failure: wait for the copies already in flight into the caller's buffers before returning the error
  auto fail = [p](int code) {
    for (auto s2 : p->streams) cudaStreamSynchronize(s2);
    return code;
  };
  int s = 0;
  for (int n0 = 0; n0 < Ng; n0 += p->chunk, s = (s + 1) % p->ns) {
    const int n = (Ng - n0 < p->chunk) ? Ng - n0 : p->chunk;
    cudaStream_t st = p->streams[s];
    cudaError_t e = cudaMemcpyAsync(p->d_in[s], in + (size_t)n0 * p->in_elems, (size_t)n * p->in_elems * sizeof(R),
                                    cudaMemcpyHostToDevice, st);
    if (e != cudaSuccess) return fail((int)e);
    oo.workspace = p->d_ws[s];
    oo.workspace_bytes = p->ws_bytes;
    rc = solve_impl<R>((const R*)p->d_in[s], (R*)p->d_out[s], ff ? (R*)p->d_ff[s] : nullptr, n, dt, dh, gamma, scheme,
                       riemann, limiter, &oo, st);
    if (rc != HYDRO_OK) return fail(rc);
    if (max_speed_host) {  // next step's CFL reduction while the chunk is still on the device: a running
      // maximum per stream over its chunks (the update's fused reduction overwrites its scalar per launch; next to the PCIe
      // copies this extra pass over `out` in HBM costs nothing measurable)
      rc = dt_impl<R>((const R*)p->d_out[s], n, 0, gamma, 0, reinterpret_cast<R*>(static_cast<double*>(p->d_speed) + s), st, true);
      if (rc != HYDRO_OK) return fail(rc);
    }
    e = cudaMemcpyAsync(out + (size_t)n0 * p->out_elems, p->d_out[s], (size_t)n * p->out_elems * sizeof(R),
                        cudaMemcpyDeviceToHost, st);
    if (e != cudaSuccess) return fail((int)e);
    if (ff) {
      e = cudaMemcpyAsync(ff + (size_t)n0 * p->ff_elems, p->d_ff[s], (size_t)n * p->ff_elems * sizeof(R),
                          cudaMemcpyDeviceToHost, st);
      if (e != cudaSuccess) return fail((int)e);
    }
  }
  for (auto st : p->streams) {
    cudaError_t e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) return (int)e;
  }
  if (status_host) {
    cudaError_t e = cudaMemcpy(status_host, p->d_status, 3 * sizeof(long long), cudaMemcpyDeviceToHost);
    if (e != cudaSuccess) return (int)e;
  }
  if (max_speed_host) {
    double h[16];
    cudaError_t e = cudaMemcpy(h, p->d_speed, p->ns * sizeof(double), cudaMemcpyDeviceToHost);
    if (e != cudaSuccess) return (int)e;
    R m = R(0);
    for (int i = 0; i < p->ns; ++i) {
      R v;
      std::memcpy(&v, &h[i], sizeof(R));
      m = (v != v || m != m) ? (R)NAN : (v > m ? v : m);
    }
    *max_speed_host = m;
  }
  return HYDRO_OK;
}
}  // namespace hydro

extern "C" {

int hydro_min_ghost(int scheme, int recon) {
  if (scheme < 0 || scheme > 2 || recon < 0 || recon > 1) return HYDRO_E_ENUM;
  return hydro::min_ghost(scheme, recon);
}

int hydro_has_fused(int precision_bytes, int scheme, int recon, int riemann) {
  if (scheme < 0 || scheme > 2 || recon < 0 || recon > 1 || riemann < 0 || riemann > 3) return 0;
  if (precision_bytes != 4 && precision_bytes != 8) return 0;
  return hydro::lean_available(precision_bytes, scheme, recon) ? 1 : 0;
}

int hydro_fused_fits(int precision_bytes, int scheme, int recon, int nghost) {
  if (!hydro_has_fused(precision_bytes, scheme, recon, 0)) return 0;
  if (nghost == 0) nghost = hydro::min_ghost(scheme, recon);
  if (nghost < hydro::min_ghost(scheme, recon) || nghost > 8) return 0;
  return hydro::lean_fits(precision_bytes, scheme, recon, nghost) ? 1 : 0;
}

size_t hydro_staged_workspace_bytes(int Ng, int precision_bytes, int scheme, int recon) {
  if (scheme < 0 || scheme > 2 || recon < 0 || recon > 1 || Ng <= 0) return 0;
  if (precision_bytes != 4 && precision_bytes != 8) return 0;
  const size_t slots = Ng < hydro::STAGED_MAX_SLOTS ? (size_t)Ng : (size_t)hydro::STAGED_MAX_SLOTS;
  return slots * hydro::staged_slot_bytes(scheme, recon, (size_t)precision_bytes);
}

size_t hydro_workspace_bytes(int Ng, int precision_bytes, int scheme, int recon) {
  if (hydro_fused_fits(precision_bytes, scheme, recon, 8)) return 0;
  return hydro_staged_workspace_bytes(Ng, precision_bytes, scheme, recon);
}

const char* hydro_strerror(int code) {
  switch (code) {
    case HYDRO_OK: return "success";
    case HYDRO_E_ENUM: return "enum argument out of range";
    case HYDRO_E_COUNT: return "negative group count";
    case HYDRO_E_NULL: return "required pointer is NULL";
    case HYDRO_E_ALIGN: return "device pointer not 16-byte aligned";
    case HYDRO_E_GHOST: return "ghost width smaller than the scheme needs (or > 8)";
    case HYDRO_E_WORKSPACE: return "staged path needs opts->workspace of hydro_workspace_bytes()";
    case HYDRO_E_VALUE: return "scalar argument out of range";
    case HYDRO_E_NOFUSED: return "no fused kernel for this variant";
    case HYDRO_E_TOOBIG: return "size beyond the fixed maximum of this no-allocation entry point (HYDRO_RTVD_NOALLOC_MAX_GROUPS)";
    default: return code > 0 ? cudaGetErrorString((cudaError_t)code) : "unknown hydro error";
  }
}

int hydro_solve_f32(const float* in, float* out, float* face_flux, int Ng, float dt, float dh, float gamma, int scheme,
                    int riemann, int limiter, const hydro_opts* opts, hydro_stream_t stream) {
  return hydro::solve_impl<float>(in, out, face_flux, Ng, dt, dh, gamma, scheme, riemann, limiter, opts, (cudaStream_t)stream);
}
int hydro_solve_f64(const double* in, double* out, double* face_flux, int Ng, double dt, double dh, double gamma, int scheme,
                    int riemann, int limiter, const hydro_opts* opts, hydro_stream_t stream) {
  return hydro::solve_impl<double>(in, out, face_flux, Ng, dt, dh, gamma, scheme, riemann, limiter, opts, (cudaStream_t)stream);
}
int hydro_solve_grid_f32(const float* grid_in, float* grid_out, int nx, int ny, int nz, int bc, float dt, float dh, float gamma,
                         int scheme, int riemann, int limiter, const hydro_opts* opts, hydro_stream_t stream) {
  return hydro::solve_grid_impl<float>(grid_in, grid_out, nx, ny, nz, bc, dt, dh, gamma, scheme, riemann, limiter, opts, (cudaStream_t)stream);
}
int hydro_solve_grid_f64(const double* grid_in, double* grid_out, int nx, int ny, int nz, int bc, double dt, double dh, double gamma,
                         int scheme, int riemann, int limiter, const hydro_opts* opts, hydro_stream_t stream) {
  return hydro::solve_grid_impl<double>(grid_in, grid_out, nx, ny, nz, bc, dt, dh, gamma, scheme, riemann, limiter, opts, (cudaStream_t)stream);
}
size_t hydro_advance_workspace_bytes(int nx, int ny, int nz, int precision_bytes, int scheme, int limiter, const hydro_opts* opts) {
  if (nx < 0 || ny < 0 || nz < 0 || nx % hydro::PS || ny % hydro::PS || nz % hydro::PS) return 0;
  if (scheme < 0 || scheme > 2 || limiter < 0 || limiter > 3) return 0;
  if (precision_bytes == 4) return hydro::advance_bytes<float>(nx, ny, nz, scheme, limiter, opts);
  if (precision_bytes == 8) return hydro::advance_bytes<double>(nx, ny, nz, scheme, limiter, opts);
  return 0;
}
int hydro_advance_f32(float* grid, int nx, int ny, int nz, int bc, int steps, float dh, float gamma, int scheme, int riemann, int limiter,
                      const hydro_opts* opts, void* work, size_t work_bytes, double* elapsed, hydro_stream_t stream) {
  return hydro::advance_impl<float>(grid, nx, ny, nz, bc, steps, dh, gamma, scheme, riemann, limiter, opts, work, work_bytes, elapsed,
                                    (cudaStream_t)stream);
}
int hydro_advance_f64(double* grid, int nx, int ny, int nz, int bc, int steps, double dh, double gamma, int scheme, int riemann,
                      int limiter, const hydro_opts* opts, void* work, size_t work_bytes, double* elapsed, hydro_stream_t stream) {
  return hydro::advance_impl<double>(grid, nx, ny, nz, bc, steps, dh, gamma, scheme, riemann, limiter, opts, work, work_bytes, elapsed,
                                     (cudaStream_t)stream);
}
int hydro_dt_f32(const float* u, int Ng, int nghost, float gamma, int norm, float* max_speed, hydro_stream_t stream) {
  return hydro::dt_impl<float>(u, Ng, nghost, gamma, norm, max_speed, (cudaStream_t)stream);
}
int hydro_dt_f64(const double* u, int Ng, int nghost, double gamma, int norm, double* max_speed, hydro_stream_t stream) {
  return hydro::dt_impl<double>(u, Ng, nghost, gamma, norm, max_speed, (cudaStream_t)stream);
}

int hydro_pipeline_create(hydro_pipeline** pp, int precision_bytes, int nghost, int groups_per_chunk, int nstreams) {
  if (!pp) return HYDRO_E_NULL;
  *pp = nullptr;
  if (precision_bytes != 4 && precision_bytes != 8) return HYDRO_E_VALUE;
  if (nghost < 2 || nghost > 8) return HYDRO_E_GHOST;
  if (groups_per_chunk < 1 || nstreams < 1 || nstreams > 16) return HYDRO_E_VALUE;
  hydro_pipeline* p = new (std::nothrow) hydro_pipeline();
  if (!p) return (int)cudaErrorMemoryAllocation;
  p->prec = precision_bytes;
  p->g = nghost;
  p->chunk = groups_per_chunk;
  p->ns = nstreams;
  const size_t S = hydro::PS + 2 * nghost;
  p->in_elems = 5 * S * S * S;
  p->out_elems = 5 * (size_t)hydro::PS * hydro::PS * hydro::PS;
  p->ff_elems = 9 * 5 * (size_t)hydro::PS * hydro::PS;
  p->ws_bytes = 0;
  p->d_status = nullptr;
  p->d_speed = nullptr;
  p->streams.assign(nstreams, nullptr);
  p->d_in.assign(nstreams, nullptr);
  p->d_out.assign(nstreams, nullptr);
  p->d_ff.assign(nstreams, nullptr);
  p->d_ws.assign(nstreams, nullptr);
  bool ok = cudaMalloc(&p->d_status, 3 * sizeof(long long)) == cudaSuccess;
  ok = ok && cudaMalloc(&p->d_speed, 16 * sizeof(double)) == cudaSuccess;
  for (int s = 0; ok && s < nstreams; ++s) {
    ok = ok && cudaStreamCreateWithFlags(&p->streams[s], cudaStreamNonBlocking) == cudaSuccess;
    ok = ok && cudaMalloc(&p->d_in[s], p->in_elems * groups_per_chunk * precision_bytes) == cudaSuccess;
    ok = ok && cudaMalloc(&p->d_out[s], p->out_elems * groups_per_chunk * precision_bytes) == cudaSuccess;
    ok = ok && cudaMalloc(&p->d_ff[s], p->ff_elems * groups_per_chunk * precision_bytes) == cudaSuccess;
  }
  if (!ok) {
    hydro_pipeline_destroy(p);
    return (int)cudaErrorMemoryAllocation;
  }
  *pp = p;
  return HYDRO_OK;
}

void hydro_pipeline_destroy(hydro_pipeline* p) {
  if (!p) return;
  for (auto s : p->streams) if (s) { cudaStreamSynchronize(s); cudaStreamDestroy(s); }
  for (auto v : {&p->d_in, &p->d_out, &p->d_ff, &p->d_ws})
    for (auto b : *v) if (b) cudaFree(b);
  if (p->d_status) cudaFree(p->d_status);
  if (p->d_speed) cudaFree(p->d_speed);
  delete p;
}

int hydro_pipeline_solve_f32(hydro_pipeline* p, const float* in, float* out, float* face_flux, int Ng, float dt, float dh,
                             float gamma, int scheme, int riemann, int limiter, const hydro_opts* opts, long long* status_host,
                             float* max_speed_host) {
  return hydro::pipeline_solve<float>(p, in, out, face_flux, Ng, dt, dh, gamma, scheme, riemann, limiter, opts, status_host,
                                      max_speed_host);
}
int hydro_pipeline_solve_f64(hydro_pipeline* p, const double* in, double* out, double* face_flux, int Ng, double dt,
                             double dh, double gamma, int scheme, int riemann, int limiter, const hydro_opts* opts,
                             long long* status_host, double* max_speed_host) {
  return hydro::pipeline_solve<double>(p, in, out, face_flux, Ng, dt, dh, gamma, scheme, riemann, limiter, opts, status_host,
                                       max_speed_host);
}

}  // extern "C"
