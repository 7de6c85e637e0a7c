// hydro_staged.cuh -- the generic "staged" solver: one CTA per patch group, one phase per
// stage of the scheme over the whole 3-D work box, intermediates (face states, fluxes) in a
// caller-supplied per-CTA global scratch slot.  This is the organisation the paper describes
// for its own kernel (one thread block per patch group, temporaries in global memory that never
// cross PCIe) and serves here as the any-variant path and as the
// bit-level cross-check of the fused z-marching kernels (same device arithmetic, hydro_math.cuh).
//
// Phases (interior coordinates, cells [0,16), ghosts negative / >= 16):
//   CTU: W -> traced face states on [-1,16]^3 -> F*_d -> transverse
//                         correction (half nu, S4) -> F_d -> update -> boundary-flux store
//   MHM: W -> untraced face states + cell-local Hancock half step -> F_d -> ...
//   VL   : W -> first-order F1_d -> U^{n+1/2} -> untraced face states -> F_d -> ...
#pragma once
#include "hydro_launch.cuh"

namespace hydro {

constexpr int STAGED_NT = 256;

template <class R> struct Box {  // inclusive bounds, interior coordinates
  int lo[3], hi[3];
  __device__ __forceinline__ int count() const {
    return (hi[0] - lo[0] + 1) * (hi[1] - lo[1] + 1) * (hi[2] - lo[2] + 1);
  }
  __device__ __forceinline__ void decode(int idx, int& i, int& j, int& k) const {
    const int nx = hi[0] - lo[0] + 1, ny = hi[1] - lo[1] + 1;
    i = lo[0] + idx % nx;
    const int r = idx / nx;
    j = lo[1] + r % ny;
    k = lo[2] + r / ny;
  }
};

// scratch view: SoA arrays of n = SW^3 elements, work box half width GW
template <class R, int GW> struct Scratch {
  static constexpr int SW = PS + 2 * GW;
  static constexpr int N = SW * SW * SW;
  R* base;
  __device__ __forceinline__ static int id(int i, int j, int k) { return ((k + GW) * SW + (j + GW)) * SW + (i + GW); }
  // array slots: 0..4 W ; 5 + (d*2+side)*5 face states (side 0 = lo, 1 = up) ; 35 + d*5 fluxes
  __device__ __forceinline__ V5<R> ld(int slot, int x) const {
    V5<R> v;
#pragma unroll
    for (int q = 0; q < 5; ++q) v[q] = base[(size_t)(slot + q) * N + x];
    return v;
  }
  __device__ __forceinline__ void st(int slot, int x, const V5<R>& v) const {
#pragma unroll
    for (int q = 0; q < 5; ++q) base[(size_t)(slot + q) * N + x] = v[q];
  }
  __device__ __forceinline__ static int slotW() { return 0; }
  __device__ __forceinline__ static int slotS(int d, int side) { return 5 + (d * 2 + side) * 5; }
  __device__ __forceinline__ static int slotF(int d) { return 35 + d * 5; }
};

template <int D> __device__ __forceinline__ int step_id(int SW) { return D == 0 ? 1 : (D == 1 ? SW : SW * SW); }

// face states of cell x along D from the primitive array in slot `src`
template <class R, int GW, int RECON, bool TRACE, int D>
__device__ __forceinline__ void recon_cell(const Scratch<R, GW>& s, int src, int x, const Par<R>& p, V5<R>& lo, V5<R>& up) {
  constexpr int st = (D == 0 ? 1 : (D == 1 ? Scratch<R, GW>::SW : Scratch<R, GW>::SW * Scratch<R, GW>::SW));
  const V5<R> W0 = to_normal<D>(s.ld(src, x));
  const V5<R> Wm1 = to_normal<D>(s.ld(src, x - st)), Wp1 = to_normal<D>(s.ld(src, x + st));
  V5<R> Wm2 = W0, Wp2 = W0;
  if (RECON == RECON_PPM) {
    Wm2 = to_normal<D>(s.ld(src, x - 2 * st));
    Wp2 = to_normal<D>(s.ld(src, x + 2 * st));
  }
  V5<R> l, u;
  reconstruct<RECON, TRACE>(Wm2, Wm1, W0, Wp1, Wp2, p, l, u);
  lo = from_normal<D>(l);
  up = from_normal<D>(u);
}

// Riemann fluxes at the lower faces of the cells of `b` along D: F[D](c) = RS(upsrc(c - e_D), losrc(c))
template <class R, int GW, int RS, int D>
__device__ __forceinline__ void flux_phase(const Scratch<R, GW>& s, int up_slot, int lo_slot, const Box<R>& b,
                                           const Par<R>& p, Cnt& c) {
  constexpr int st = (D == 0 ? 1 : (D == 1 ? Scratch<R, GW>::SW : Scratch<R, GW>::SW * Scratch<R, GW>::SW));
  const int n = b.count();
  for (int idx = threadIdx.x; idx < n; idx += STAGED_NT) {
    int i, j, k;
    b.decode(idx, i, j, k);
    const int x = s.id(i, j, k);
    const V5<R> f = riemann_d<RS, D>(s.ld(up_slot, x - st), s.ld(lo_slot, x), p, c);
    s.st(s.slotF(D), x, f);
  }
}

template <class R, int GW, int RECON, bool TRACE, int D>
__device__ __forceinline__ void recon_phase(const Scratch<R, GW>& s, int src, const Box<R>& b, const Par<R>& p) {
  const int n = b.count();
  for (int idx = threadIdx.x; idx < n; idx += STAGED_NT) {
    int i, j, k;
    b.decode(idx, i, j, k);
    const int x = s.id(i, j, k);
    V5<R> lo, up;
    recon_cell<R, GW, RECON, TRACE, D>(s, src, x, p, lo, up);
    s.st(s.slotS(D, 0), x, lo);
    s.st(s.slotS(D, 1), x, up);
  }
}

// CTU transverse correction of both face states of direction D (S4: half nu, cyclic t1,t2)
template <class R, int GW, int D>
__device__ __forceinline__ void ctu_correct_phase(const Scratch<R, GW>& s, const Par<R>& p, Cnt& c) {
  constexpr int SW = Scratch<R, GW>::SW;
  constexpr int T1 = (D + 1) % 3, T2 = (D + 2) % 3;
  constexpr int st1 = (T1 == 0 ? 1 : (T1 == 1 ? SW : SW * SW)), st2 = (T2 == 0 ? 1 : (T2 == 1 ? SW : SW * SW));
  Box<R> b;
  for (int a = 0; a < 3; ++a) {
    b.lo[a] = (a == D) ? -1 : 0;
    b.hi[a] = (a == D) ? PS : PS - 1;
  }
  const int n = b.count();
  for (int idx = threadIdx.x; idx < n; idx += STAGED_NT) {
    int i, j, k;
    b.decode(idx, i, j, k);
    const int x = s.id(i, j, k);
    const V5<R> A1 = s.ld(s.slotF(T1), x + st1), A0 = s.ld(s.slotF(T1), x);
    const V5<R> B1 = s.ld(s.slotF(T2), x + st2), B0 = s.ld(s.slotF(T2), x);
    V5<R> dq;
#pragma unroll
    for (int q = 0; q < 5; ++q) dq[q] = p.hnu * ((A1[q] - A0[q]) + (B1[q] - B0[q]));
#pragma unroll
    for (int side = 0; side < 2; ++side) {
      V5<R> U = prim2cons(s.ld(s.slotS(D, side), x), p);
#pragma unroll
      for (int q = 0; q < 5; ++q) U[q] = U[q] - dq[q];
      s.st(s.slotS(D, side), x, cons2prim(U, p, c));
    }
  }
}

template <class R> __device__ __forceinline__ V5<R> load_in(const R* in, size_t nS, int xin) {
  V5<R> U;
#pragma unroll
  for (int q = 0; q < 5; ++q) U[q] = __ldg(in + q * nS + xin);
  return U;
}

template <class R, int SCHEME, int RECON, int RS>
__global__ void __launch_bounds__(STAGED_NT) staged_kernel(const R* __restrict__ in, R* __restrict__ out,
                                                           R* __restrict__ face_flux, int Ng, int g, Par<R> p,
                                                           const R* __restrict__ max_speed, R cfl,
                                                           long long* status, R* scratch) {
  apply_device_dt(p, max_speed, cfl);
  constexpr int GW = (SCHEME == SCHEME_VL ? 3 : 2) + (RECON == RECON_PPM ? 1 : 0);
  using Sc = Scratch<R, GW>;
  Sc s;
  s.base = scratch + (size_t)blockIdx.x * 50 * Sc::N;
  const int S = PS + 2 * g;
  const size_t nS = (size_t)S * S * S;
  Cnt c = {0, 0, 0};

  for (int grp = blockIdx.x; grp < Ng; grp += gridDim.x) {
    const R* gin = in + (size_t)grp * 5 * nS;
    // ---- (1) primitive variables on the work box
    for (int idx = threadIdx.x; idx < Sc::N; idx += STAGED_NT) {
      const int i = idx % Sc::SW - GW, r = idx / Sc::SW, j = r % Sc::SW - GW, k = r / Sc::SW - GW;
      const int xin = ((k + g) * S + (j + g)) * S + (i + g);
      s.st(Sc::slotW(), idx, cons2prim(load_in(gin, nS, xin), p, c));
    }
    __syncthreads();
    Box<R> b;
    if (SCHEME == SCHEME_CTU) {
      for (int a = 0; a < 3; ++a) { b.lo[a] = -1; b.hi[a] = PS; }
      recon_phase<R, GW, RECON, true, 0>(s, Sc::slotW(), b, p);
      recon_phase<R, GW, RECON, true, 1>(s, Sc::slotW(), b, p);
      recon_phase<R, GW, RECON, true, 2>(s, Sc::slotW(), b, p);
      __syncthreads();
      // F*_d: faces f_d in [0,16], transverse in [-1,16]
      b.lo[0] = 0; flux_phase<R, GW, RS, 0>(s, Sc::slotS(0, 1), Sc::slotS(0, 0), b, p, c); b.lo[0] = -1;
      b.lo[1] = 0; flux_phase<R, GW, RS, 1>(s, Sc::slotS(1, 1), Sc::slotS(1, 0), b, p, c); b.lo[1] = -1;
      b.lo[2] = 0; flux_phase<R, GW, RS, 2>(s, Sc::slotS(2, 1), Sc::slotS(2, 0), b, p, c); b.lo[2] = -1;
      __syncthreads();
      ctu_correct_phase<R, GW, 0>(s, p, c);
      ctu_correct_phase<R, GW, 1>(s, p, c);
      ctu_correct_phase<R, GW, 2>(s, p, c);
      __syncthreads();
    } else if (SCHEME == SCHEME_MHM) {
      // untraced face states of all three directions + one cell-local half-step increment (S13)
      for (int a = 0; a < 3; ++a) { b.lo[a] = -1; b.hi[a] = PS; }
      const int n = b.count();
      for (int idx = threadIdx.x; idx < n; idx += STAGED_NT) {
        int i, j, k;
        b.decode(idx, i, j, k);
        const int x = s.id(i, j, k);
        V5<R> lo[3], up[3];
        recon_cell<R, GW, RECON, false, 0>(s, Sc::slotW(), x, p, lo[0], up[0]);
        recon_cell<R, GW, RECON, false, 1>(s, Sc::slotW(), x, p, lo[1], up[1]);
        recon_cell<R, GW, RECON, false, 2>(s, Sc::slotW(), x, p, lo[2], up[2]);
        V5<R> dF[3];
        {
          const V5<R> fu = from_normal<0>(phys_flux(to_normal<0>(up[0]), p)), fl = from_normal<0>(phys_flux(to_normal<0>(lo[0]), p));
#pragma unroll
          for (int q = 0; q < 5; ++q) dF[0][q] = fu[q] - fl[q];
        }
        {
          const V5<R> fu = from_normal<1>(phys_flux(to_normal<1>(up[1]), p)), fl = from_normal<1>(phys_flux(to_normal<1>(lo[1]), p));
#pragma unroll
          for (int q = 0; q < 5; ++q) dF[1][q] = fu[q] - fl[q];
        }
        {
          const V5<R> fu = from_normal<2>(phys_flux(to_normal<2>(up[2]), p)), fl = from_normal<2>(phys_flux(to_normal<2>(lo[2]), p));
#pragma unroll
          for (int q = 0; q < 5; ++q) dF[2][q] = fu[q] - fl[q];
        }
        V5<R> inc;
#pragma unroll
        for (int q = 0; q < 5; ++q) inc[q] = p.hnu * ((dF[0][q] + dF[1][q]) + dF[2][q]);
        const bool in_i = (i >= 0 && i < PS), in_j = (j >= 0 && j < PS), in_k = (k >= 0 && k < PS);
        const bool need[3] = {in_j && in_k, in_i && in_k, in_i && in_j};  // transverse coordinates interior
#pragma unroll
        for (int d = 0; d < 3; ++d) {
          if (!need[d]) continue;
#pragma unroll
          for (int side = 0; side < 2; ++side) {
            V5<R> U = prim2cons(side ? up[d] : lo[d], p);
#pragma unroll
            for (int q = 0; q < 5; ++q) U[q] = U[q] - inc[q];
            s.st(Sc::slotS(d, side), x, cons2prim(U, p, c));
          }
        }
      }
      __syncthreads();
    } else {  // VL
      constexpr int H = GW - 1;  // half-step state needed on [-H, 16+H)^3
      for (int a = 0; a < 3; ++a) { b.lo[a] = -H; b.hi[a] = PS + H - 1; }
      b.hi[0] = PS + H; flux_phase<R, GW, RS, 0>(s, Sc::slotW(), Sc::slotW(), b, p, c); b.hi[0] = PS + H - 1;
      b.hi[1] = PS + H; flux_phase<R, GW, RS, 1>(s, Sc::slotW(), Sc::slotW(), b, p, c); b.hi[1] = PS + H - 1;
      b.hi[2] = PS + H; flux_phase<R, GW, RS, 2>(s, Sc::slotW(), Sc::slotW(), b, p, c); b.hi[2] = PS + H - 1;
      __syncthreads();
      {
        const int n = b.count();
        for (int idx = threadIdx.x; idx < n; idx += STAGED_NT) {
          int i, j, k;
          b.decode(idx, i, j, k);
          const int x = s.id(i, j, k);
          const int xin = ((k + g) * S + (j + g)) * S + (i + g);
          V5<R> U = load_in(gin, nS, xin);
          const V5<R> fx1 = s.ld(Sc::slotF(0), x + 1), fx0 = s.ld(Sc::slotF(0), x);
          const V5<R> fy1 = s.ld(Sc::slotF(1), x + Sc::SW), fy0 = s.ld(Sc::slotF(1), x);
          const V5<R> fz1 = s.ld(Sc::slotF(2), x + Sc::SW * Sc::SW), fz0 = s.ld(Sc::slotF(2), x);
#pragma unroll
          for (int q = 0; q < 5; ++q) U[q] = U[q] - p.hnu * (((fx1[q] - fx0[q]) + (fy1[q] - fy0[q])) + (fz1[q] - fz0[q]));
          s.st(Sc::slotW(), x, cons2prim(U, p, c));  // W^{n+1/2} replaces W^n (W^n is not read again)
        }
      }
      __syncthreads();
      for (int a = 0; a < 3; ++a) { b.lo[a] = 0; b.hi[a] = PS - 1; }
      b.lo[0] = -1; b.hi[0] = PS; recon_phase<R, GW, RECON, false, 0>(s, Sc::slotW(), b, p); b.lo[0] = 0; b.hi[0] = PS - 1;
      b.lo[1] = -1; b.hi[1] = PS; recon_phase<R, GW, RECON, false, 1>(s, Sc::slotW(), b, p); b.lo[1] = 0; b.hi[1] = PS - 1;
      b.lo[2] = -1; b.hi[2] = PS; recon_phase<R, GW, RECON, false, 2>(s, Sc::slotW(), b, p);
      __syncthreads();
    }
    // ---- final fluxes F_d: f_d in [0,16], transverse in [0,16)
    for (int a = 0; a < 3; ++a) { b.lo[a] = 0; b.hi[a] = PS - 1; }
    b.hi[0] = PS; flux_phase<R, GW, RS, 0>(s, Sc::slotS(0, 1), Sc::slotS(0, 0), b, p, c); b.hi[0] = PS - 1;
    b.hi[1] = PS; flux_phase<R, GW, RS, 1>(s, Sc::slotS(1, 1), Sc::slotS(1, 0), b, p, c); b.hi[1] = PS - 1;
    b.hi[2] = PS; flux_phase<R, GW, RS, 2>(s, Sc::slotS(2, 1), Sc::slotS(2, 0), b, p, c); b.hi[2] = PS - 1;
    __syncthreads();
    // ---- conservative update and patch-boundary flux store
    R* gout = out + (size_t)grp * 5 * PS * PS * PS;
    for (int idx = threadIdx.x; idx < PS * PS * PS; idx += STAGED_NT) {
      const int i = idx % PS, j = (idx / PS) % PS, k = idx / (PS * PS);
      const int x = s.id(i, j, k);
      const int xin = ((k + g) * S + (j + g)) * S + (i + g);
      V5<R> U = load_in(gin, nS, xin);
      const V5<R> fx1 = s.ld(Sc::slotF(0), x + 1), fx0 = s.ld(Sc::slotF(0), x);
      const V5<R> fy1 = s.ld(Sc::slotF(1), x + Sc::SW), fy0 = s.ld(Sc::slotF(1), x);
      const V5<R> fz1 = s.ld(Sc::slotF(2), x + Sc::SW * Sc::SW), fz0 = s.ld(Sc::slotF(2), x);
#pragma unroll
      for (int q = 0; q < 5; ++q) U[q] = U[q] - p.nu * (((fx1[q] - fx0[q]) + (fy1[q] - fy0[q])) + (fz1[q] - fz0[q]));
      const V5<R> Wn = cons2prim(U, p, c);
      if (p.min_dens > R(0) || p.min_pres > R(0)) U = prim2cons(Wn, p);
#pragma unroll
      for (int q = 0; q < 5; ++q) gout[q * PS * PS * PS + idx] = U[q];
    }
    if (face_flux) {
      R* gff = face_flux + (size_t)grp * 9 * 5 * PS * PS;
      for (int idx = threadIdx.x; idx < 9 * 5 * PS * PS; idx += STAGED_NT) {
        const int a = idx % PS, bb = (idx / PS) % PS, q = (idx / (PS * PS)) % 5, pl = idx / (5 * PS * PS);
        const int d = pl / 3, f = 8 * (pl % 3);
        // in-plane order: d=x -> [k][j], d=y -> [k][i], d=z -> [j][i]
        const int i = d == 0 ? f : a, j = d == 0 ? a : (d == 1 ? f : bb), k = d == 2 ? f : bb;
        gff[idx] = s.base[(size_t)(Sc::slotF(d) + q) * Sc::N + s.id(i, j, k)];
      }
    }
    __syncthreads();  // scratch is reused by the next group of this CTA
  }
  flush_counters(c, status);
}

template <class R, int SCHEME, int RECON, int RS> cudaError_t launch_staged(const SolveArgs<R>& a) {
  const size_t slot = staged_slot_bytes(SCHEME, RECON, sizeof(R));
  size_t slots = a.workspace_bytes / slot;
  if (slots > (size_t)a.Ng) slots = a.Ng;
  if (slots > (size_t)STAGED_MAX_SLOTS) slots = STAGED_MAX_SLOTS;
  staged_kernel<R, SCHEME, RECON, RS><<<(unsigned)slots, STAGED_NT, 0, a.stream>>>(
      a.in, a.out, a.face_flux, a.Ng, a.g, a.par, a.max_speed, a.cfl, a.status, static_cast<R*>(a.workspace));
  return cudaGetLastError();
}

}  // namespace hydro
