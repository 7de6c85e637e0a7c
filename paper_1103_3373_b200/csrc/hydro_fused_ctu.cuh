// hydro_fused_ctu.cuh -- fused z-marching CTU kernel (steps (1)-(5) in one launch,
// every intermediate on chip).
//
// One persistent CTA per SM slot walks its patch groups; inside a group it marches along z.
// Thread (ii, jj) of the 18 x 18 tile owns the column (i, j) = (ii-1, jj-1) in [-1,16]^2, i.e. the
// interior plus the one-cell ring whose traced states / first-pass fluxes the transverse correction
// of the interior needs.  Everything along z is column-local and is carried from
// plane to plane in registers (or per-thread shared-memory slots, template mask SM): the traced z
// states, F*_z at the two faces of the current plane, the corrected upper z state of the previous plane,
// the final F_z below the previous plane and that plane's x+y flux difference.  Along x and y,
// neighbours exchange 5-vectors through four shared-memory buffers (up states, F*_x/F*_y, corrected
// up states, F_x/F_y): 5 CTA barriers per plane.
//
// Input planes arrive by 1-D bulk async copies (cp.async.bulk + mbarrier, i.e. TMA without a tensor
// map: rows of 16+2g cells are not 16-byte multiples for g = 3, whole z planes always are), two planes
// in flight, continuing across group boundaries so the first planes of the next group are already
// resident when the current one finishes.  Primitive planes live in a (2 RW + 1)-deep ring.
//
// Iteration t (plane index, t = -GW-LA .. 16; most work for t in [-1,16]):
//   A  convert raw plane t+LA to primitive (ring), prefetch U(t-1) for the update          | barrier
//   B  z: traced states of plane t+1 (column-local), F*_z(t+1) = RS(up_z(t), lo_z(t+1))
//   C  x,y: traced states of plane t -> up states to the exchange buffers                 | barrier
//   D  F*_x(t), F*_y(t) -> exchange buffers                                                | barrier
//   E  transverse correction of the six face states of plane t (half nu, S4)               | barrier
//   F  F_x(t), F_y(t), F_z(t) = RS(up_z'(t-1), lo_z'(t)); patch-boundary flux store        | barrier
//   G  x+y flux difference of plane t; conservative update + store of plane t-1
#pragma once
#include <cstdint>
#include "hydro_launch.cuh"
#include "hydro_ptx.cuh"

namespace hydro {

constexpr int FT = PS + 2;          // tile side: interior + one-cell ring
constexpr int FCOL = FUSED_COLS;    // 324 columns
constexpr int FNT = FUSED_NT;       // threads per CTA (11 warps)

// ---- per-thread 5-vector that lives either in registers or in a private shared-memory slot --------
template <class R, bool SM> struct P5;
template <class R> struct P5<R, false> {
  V5<R> v;
  __device__ __forceinline__ void bind(R*) {}
  __device__ __forceinline__ V5<R> get() const { return v; }
  __device__ __forceinline__ void set(const V5<R>& x) { v = x; }
};
template <class R> struct P5<R, true> {
  R* p;
  __device__ __forceinline__ void bind(R* slot) { p = slot + threadIdx.x; }
  __device__ __forceinline__ V5<R> get() const {
    V5<R> x;
#pragma unroll
    for (int q = 0; q < 5; ++q) x[q] = p[q * FNT];
    return x;
  }
  __device__ __forceinline__ void set(const V5<R>& x) {
#pragma unroll
    for (int q = 0; q < 5; ++q) p[q * FNT] = x[q];
  }
};
// double-buffered variant: `nxt` is produced one plane ahead of its use as `cur`
template <class R, bool SM> struct DB5;
template <class R> struct DB5<R, false> {
  V5<R> c, n;
  __device__ __forceinline__ void bind(R*, R*) {}
  __device__ __forceinline__ V5<R> cur() const { return c; }
  __device__ __forceinline__ V5<R> nxt() const { return n; }
  __device__ __forceinline__ void set_nxt(const V5<R>& x) { n = x; }
  __device__ __forceinline__ void advance() { c = n; }
};
template <class R> struct DB5<R, true> {
  R *pc, *pn;
  __device__ __forceinline__ void bind(R* a, R* b) { pc = a + threadIdx.x; pn = b + threadIdx.x; }
  __device__ __forceinline__ V5<R> cur() const {
    V5<R> x;
#pragma unroll
    for (int q = 0; q < 5; ++q) x[q] = pc[q * FNT];
    return x;
  }
  __device__ __forceinline__ V5<R> nxt() const {
    V5<R> x;
#pragma unroll
    for (int q = 0; q < 5; ++q) x[q] = pn[q * FNT];
    return x;
  }
  __device__ __forceinline__ void set_nxt(const V5<R>& x) {
#pragma unroll
    for (int q = 0; q < 5; ++q) pn[q * FNT] = x[q];
  }
  __device__ __forceinline__ void advance() { R* t = pc; pc = pn; pn = t; }
};

template <class R, int RECON, int SM> struct CtuCfg {
  static constexpr int GW = 2 + RECON;       // ghost cells read
  static constexpr int RW = 1 + RECON;       // reconstruction half width
  static constexpr int LA = RW + 1;          // plane look-ahead of the conversion stage
  static constexpr int SWP = PS + 2 * GW;    // primitive plane side
  static constexpr int NW = 2 * RW + 1;      // primitive ring depth
  static constexpr int NPL = PS + 2 * GW;    // planes consumed per group
  // shared-memory carve-up: mbarriers | raw planes [2][5][S*S] | W ring | 4 exchange buffers | private slots
  static size_t smem_bytes(int g) { return ctu_smem_bytes(sizeof(R), RECON, g, SM); }
};

template <class R, int RECON, int RS, int SM, int MINB>
__global__ void __launch_bounds__(FNT, MINB)
ctu_fused_kernel(const R* __restrict__ in, R* __restrict__ out, R* __restrict__ face_flux, int Ng, int g, Par<R> p,
                 const R* __restrict__ max_speed, R cfl, long long* status) {
  using C = CtuCfg<R, RECON, SM>;
  constexpr int GW = C::GW, RW = C::RW, LA = C::LA, SWP = C::SWP, NW = C::NW, NPL = C::NPL;
  constexpr int WPL = SWP * SWP;  // cells per primitive plane
  apply_device_dt(p, max_speed, cfl);

  const int S = PS + 2 * g;
  const int SS = S * S;
  const size_t nS = (size_t)SS * S;
  const int off = g - GW;  // unused outer ghost layers

  extern __shared__ __align__(16) unsigned char smem[];
  uint64_t* bar = reinterpret_cast<uint64_t*>(smem);
  R* raw = reinterpret_cast<R*>(smem + 16);          // [2][5][SS]
  R* ring = raw + (size_t)2 * 5 * SS;                // [NW][5][WPL]
  R* ex = ring + (size_t)NW * 5 * WPL;               // [4][5][FCOL]
  R* slots = ex + (size_t)4 * 5 * FCOL;              // [nslots][5][FNT]
  R* exA = ex;
  R* exB = ex + 5 * FCOL;
  R* exC = ex + 10 * FCOL;
  R* exD = ex + 15 * FCOL;

  const int tid = threadIdx.x;
  const bool active = tid < FCOL;
  const int ii = tid % FT, jj = tid / FT;            // tile coordinates; cell (i,j) = (ii-1, jj-1)
  const bool in_i = active && ii >= 1 && ii <= PS, in_j = active && jj >= 1 && jj <= PS;
  const bool interior = in_i && in_j;
  const int wb = (jj + GW - 1) * SWP + (ii + GW - 1);  // own index in a primitive plane

  // per-thread carried state
  DB5<R, (SM & SM_Z) != 0> zlo, zup;      // traced z states of planes t (cur) and t+1 (nxt)
  DB5<R, (SM & SM_F1Z) != 0> f1z;         // F*_z at faces t (cur) and t+1 (nxt)
  P5<R, (SM & SM_CARRY) != 0> uzc, f2z, sxy;  // corrected up_z of plane t-1; F_z at face t-1 -> t; (dFx+dFy) of plane t-1
  P5<R, (SM & SM_XY) != 0> lox, loy, upx, upy, loz;  // x/y states between stages C..F, corrected lo_z E..F
  {
    R* s = slots;
    auto take = [&]() { R* r = s; s += 5 * FNT; return r; };
    if (SM & SM_Z) { R* a = take(); R* b = take(); zlo.bind(a, b); a = take(); b = take(); zup.bind(a, b); }
    if (SM & SM_F1Z) { R* a = take(); R* b = take(); f1z.bind(a, b); }
    if (SM & SM_CARRY) { uzc.bind(take()); f2z.bind(take()); sxy.bind(take()); }
    if (SM & SM_XY) { lox.bind(take()); loy.bind(take()); upx.bind(take()); upy.bind(take()); loz.bind(take()); }
  }

  // ---- plane pipeline: sequence number n = m * NPL + (plane + GW) over this CTA's groups m
  const int my_groups = (Ng - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x;
  const int total_planes = my_groups * NPL;
  const uint32_t plane_bytes = (uint32_t)(5 * SS * sizeof(R));
  auto issue = [&](int n) {  // called by thread 0 only
    if (n >= total_planes) return;
    const int m = n / NPL, pl = n % NPL;               // pl = plane + GW
    const size_t grp = (size_t)blockIdx.x + (size_t)m * gridDim.x;
    const R* src = in + grp * 5 * nS + (size_t)(pl + off) * SS;
    uint64_t* b = bar + (n & 1);
    R* dst = raw + (size_t)(n & 1) * 5 * SS;
    mbar_expect_tx(b, plane_bytes);
#pragma unroll
    for (int q = 0; q < 5; ++q) bulk_g2s(dst + (size_t)q * SS, src + q * nS, (uint32_t)(SS * sizeof(R)), b);
  };
  if (tid == 0) {
    mbar_init(bar, 1);
    mbar_init(bar + 1, 1);
    fence_mbar_init();
    fence_async_smem();
  }
  __syncthreads();
  if (tid == 0) { issue(0); issue(1); }

  Cnt c = {0, 0, 0};
  int nseq = 0;  // next plane sequence number to convert

  for (int m = 0; m < my_groups; ++m) {
    const size_t grp = (size_t)blockIdx.x + (size_t)m * gridDim.x;
    const R* gin = in + grp * 5 * nS;
    R* gout = out + grp * 5 * PS * PS * PS;
    R* gff = face_flux ? face_flux + grp * 9 * 5 * PS * PS : nullptr;

    for (int t = -GW - LA; t <= PS; ++t) {
      // ================= A: convert plane t+LA; prefetch U(t-1) =================
      const int pc = t + LA;
      if (pc <= PS - 1 + GW) {  // pc >= -GW by construction of the loop start
        const int st = nseq & 1;
        while (!mbar_try_wait(bar + st, (uint32_t)((nseq >> 1) & 1))) {}
        const R* rp = raw + (size_t)st * 5 * SS;
        R* wp = ring + (size_t)((pc + GW) % NW) * 5 * WPL;
        for (int idx = tid; idx < WPL; idx += FNT) {
          const int a = idx % SWP, b = idx / SWP;
          const int src = (b + off) * S + (a + off);
          V5<R> U;
#pragma unroll
          for (int q = 0; q < 5; ++q) U[q] = rp[q * SS + src];
          const V5<R> W = cons2prim(U, p, c);
#pragma unroll
          for (int q = 0; q < 5; ++q) wp[q * WPL + idx] = W[q];
        }
      }
      V5<R> Uold;
      const bool do_upd = interior && t >= 1;  // update of plane t-1 in [0,16)
      if (do_upd) {
        const int xin = ((t - 1 + g) * S + (jj - 1 + g)) * S + (ii - 1 + g);
#pragma unroll
        for (int q = 0; q < 5; ++q) Uold[q] = __ldg(gin + q * nS + xin);
      }
      __syncthreads();  // S1: primitive plane visible; raw stage consumed
      if (pc <= PS - 1 + GW) {
        if (tid == 0) { fence_async_smem(); issue(nseq + 2); }
        ++nseq;
      }
      if (t < -2) continue;  // pipeline fill: only conversions so far (uniform over the CTA)

      // ================= B: z states of plane t+1, F*_z(t+1) =================
      const int kz = t + 1;
      if (active && kz <= PS) {
        V5<R> Wz[2 * RW + 1];
#pragma unroll
        for (int s = 0; s < 2 * RW + 1; ++s) {
          const R* wp = ring + (size_t)((kz - RW + s + GW) % NW) * 5 * WPL + wb;
          V5<R> w;
#pragma unroll
          for (int q = 0; q < 5; ++q) w[q] = wp[q * WPL];
          Wz[s] = to_normal<2>(w);
        }
        V5<R> l, u;
        reconstruct<RECON, true>(Wz[0], Wz[RW - 1], Wz[RW], Wz[RW + 1], Wz[2 * RW], p, l, u);
        const V5<R> lz = from_normal<2>(l), uz = from_normal<2>(u);
        if (kz >= 0) f1z.set_nxt(riemann_d<RS, 2>(zup.cur(), lz, p, c));
        zlo.set_nxt(lz);
        zup.set_nxt(uz);
      }
      if (t < -1) {  // t == -2: nothing else to do for this plane
        zlo.advance(); zup.advance(); f1z.advance();
        continue;
      }

      // ================= C: x,y traced states of plane t =================
      const R* wt = ring + (size_t)((t + GW) % NW) * 5 * WPL + wb;
      if (active) {
        V5<R> W0, Wa, Wb, Wc, Wd;
#pragma unroll
        for (int q = 0; q < 5; ++q) W0[q] = wt[q * WPL];
        {
#pragma unroll
          for (int q = 0; q < 5; ++q) { Wb[q] = wt[q * WPL - 1]; Wc[q] = wt[q * WPL + 1]; }
          if (RECON == RECON_PPM) {
#pragma unroll
            for (int q = 0; q < 5; ++q) { Wa[q] = wt[q * WPL - 2]; Wd[q] = wt[q * WPL + 2]; }
          } else { Wa = Wb; Wd = Wc; }
          V5<R> l, u;
          reconstruct<RECON, true>(to_normal<0>(Wa), to_normal<0>(Wb), to_normal<0>(W0), to_normal<0>(Wc), to_normal<0>(Wd), p, l, u);
          const V5<R> ux = from_normal<0>(u);
          lox.set(from_normal<0>(l));
          upx.set(ux);
#pragma unroll
          for (int q = 0; q < 5; ++q) exA[q * FCOL + tid] = ux[q];
        }
        {
#pragma unroll
          for (int q = 0; q < 5; ++q) { Wb[q] = wt[q * WPL - SWP]; Wc[q] = wt[q * WPL + SWP]; }
          if (RECON == RECON_PPM) {
#pragma unroll
            for (int q = 0; q < 5; ++q) { Wa[q] = wt[q * WPL - 2 * SWP]; Wd[q] = wt[q * WPL + 2 * SWP]; }
          } else { Wa = Wb; Wd = Wc; }
          V5<R> l, u;
          reconstruct<RECON, true>(to_normal<1>(Wa), to_normal<1>(Wb), to_normal<1>(W0), to_normal<1>(Wc), to_normal<1>(Wd), p, l, u);
          const V5<R> uy = from_normal<1>(u);
          loy.set(from_normal<1>(l));
          upy.set(uy);
#pragma unroll
          for (int q = 0; q < 5; ++q) exB[q * FCOL + tid] = uy[q];
        }
      }
      __syncthreads();  // S2

      // ================= D: F*_x(t), F*_y(t) =================
      V5<R> f1x, f1y;
      if (active && ii >= 1) {
        V5<R> ul;
#pragma unroll
        for (int q = 0; q < 5; ++q) ul[q] = exA[q * FCOL + tid - 1];
        f1x = riemann_d<RS, 0>(ul, lox.get(), p, c);
#pragma unroll
        for (int q = 0; q < 5; ++q) exC[q * FCOL + tid] = f1x[q];
      }
      if (active && jj >= 1) {
        V5<R> ul;
#pragma unroll
        for (int q = 0; q < 5; ++q) ul[q] = exB[q * FCOL + tid - FT];
        f1y = riemann_d<RS, 1>(ul, loy.get(), p, c);
#pragma unroll
        for (int q = 0; q < 5; ++q) exD[q * FCOL + tid] = f1y[q];
      }
      __syncthreads();  // S3

      // ================= E: transverse correction (half nu, cyclic t1,t2: S4) =================
      const bool plane_in = (t >= 0 && t < PS);
      V5<R> uzc_new;
      {
        V5<R> dFx, dFy, dFz;  // flux differences across this cell
        if (in_i) {
#pragma unroll
          for (int q = 0; q < 5; ++q) dFx[q] = exC[q * FCOL + tid + 1] - f1x[q];
        }
        if (in_j) {
#pragma unroll
          for (int q = 0; q < 5; ++q) dFy[q] = exD[q * FCOL + tid + FT] - f1y[q];
        }
        if (plane_in && active) {
          const V5<R> a = f1z.nxt(), b = f1z.cur();
#pragma unroll
          for (int q = 0; q < 5; ++q) dFz[q] = a[q] - b[q];
        }
        if (in_j && plane_in) {  // x states: t1 = y, t2 = z
          V5<R> dq;
#pragma unroll
          for (int q = 0; q < 5; ++q) dq[q] = p.hnu * (dFy[q] + dFz[q]);
          V5<R> U = prim2cons(lox.get(), p);
#pragma unroll
          for (int q = 0; q < 5; ++q) U[q] = U[q] - dq[q];
          lox.set(cons2prim(U, p, c));
          U = prim2cons(upx.get(), p);
#pragma unroll
          for (int q = 0; q < 5; ++q) U[q] = U[q] - dq[q];
          const V5<R> w = cons2prim(U, p, c);
#pragma unroll
          for (int q = 0; q < 5; ++q) exA[q * FCOL + tid] = w[q];
        }
        if (in_i && plane_in) {  // y states: t1 = z, t2 = x
          V5<R> dq;
#pragma unroll
          for (int q = 0; q < 5; ++q) dq[q] = p.hnu * (dFz[q] + dFx[q]);
          V5<R> U = prim2cons(loy.get(), p);
#pragma unroll
          for (int q = 0; q < 5; ++q) U[q] = U[q] - dq[q];
          loy.set(cons2prim(U, p, c));
          U = prim2cons(upy.get(), p);
#pragma unroll
          for (int q = 0; q < 5; ++q) U[q] = U[q] - dq[q];
          const V5<R> w = cons2prim(U, p, c);
#pragma unroll
          for (int q = 0; q < 5; ++q) exB[q * FCOL + tid] = w[q];
        }
        if (interior) {  // z states: t1 = x, t2 = y ; every plane t in [-1,16]
          V5<R> dq;
#pragma unroll
          for (int q = 0; q < 5; ++q) dq[q] = p.hnu * (dFx[q] + dFy[q]);
          V5<R> U = prim2cons(zlo.cur(), p);
#pragma unroll
          for (int q = 0; q < 5; ++q) U[q] = U[q] - dq[q];
          loz.set(cons2prim(U, p, c));
          U = prim2cons(zup.cur(), p);
#pragma unroll
          for (int q = 0; q < 5; ++q) U[q] = U[q] - dq[q];
          uzc_new = cons2prim(U, p, c);
        }
      }
      __syncthreads();  // S4

      // ================= F: final fluxes of plane t + boundary-flux store ============
      V5<R> f2x, f2y, f2z_new;
      const bool do_fx = plane_in && in_j && active && ii >= 1;
      const bool do_fy = plane_in && in_i && active && jj >= 1;
      if (do_fx) {
        V5<R> ul;
#pragma unroll
        for (int q = 0; q < 5; ++q) ul[q] = exA[q * FCOL + tid - 1];
        f2x = riemann_d<RS, 0>(ul, lox.get(), p, c);
#pragma unroll
        for (int q = 0; q < 5; ++q) exC[q * FCOL + tid] = f2x[q];
        if (gff && ((ii - 1) & 7) == 0) {
          R* d = gff + (size_t)(((ii - 1) >> 3) * 5) * 256 + t * PS + (jj - 1);
#pragma unroll
          for (int q = 0; q < 5; ++q) d[q * 256] = f2x[q];
        }
      }
      if (do_fy) {
        V5<R> ul;
#pragma unroll
        for (int q = 0; q < 5; ++q) ul[q] = exB[q * FCOL + tid - FT];
        f2y = riemann_d<RS, 1>(ul, loy.get(), p, c);
#pragma unroll
        for (int q = 0; q < 5; ++q) exD[q * FCOL + tid] = f2y[q];
        if (gff && ((jj - 1) & 7) == 0) {
          R* d = gff + (size_t)((3 + ((jj - 1) >> 3)) * 5) * 256 + t * PS + (ii - 1);
#pragma unroll
          for (int q = 0; q < 5; ++q) d[q * 256] = f2y[q];
        }
      }
      if (interior) {
        if (t >= 0) {
          f2z_new = riemann_d<RS, 2>(uzc.get(), loz.get(), p, c);
          if (gff && (t & 7) == 0) {
            R* d = gff + (size_t)((6 + (t >> 3)) * 5) * 256 + (jj - 1) * PS + (ii - 1);
#pragma unroll
            for (int q = 0; q < 5; ++q) d[q * 256] = f2z_new[q];
          }
        }
        uzc.set(uzc_new);
      }
      __syncthreads();  // S5

      // ================= G: conservative update of plane t-1; x+y flux difference of plane t =========
      if (interior) {
        if (do_upd) {
          const V5<R> sp = sxy.get(), fzo = f2z.get();
          V5<R> U;
#pragma unroll
          for (int q = 0; q < 5; ++q) U[q] = Uold[q] - p.nu * (sp[q] + (f2z_new[q] - fzo[q]));
          const V5<R> Wn = cons2prim(U, p, c);
          if (p.min_dens > R(0) || p.min_pres > R(0)) U = prim2cons(Wn, p);
          R* d = gout + ((t - 1) * PS + (jj - 1)) * PS + (ii - 1);
#pragma unroll
          for (int q = 0; q < 5; ++q) d[q * PS * PS * PS] = U[q];
        }
        if (t >= 0) f2z.set(f2z_new);
        if (plane_in) {
          V5<R> s;
#pragma unroll
          for (int q = 0; q < 5; ++q) s[q] = (exC[q * FCOL + tid + 1] - f2x[q]) + (exD[q * FCOL + tid + FT] - f2y[q]);
          sxy.set(s);
        }
      }
      zlo.advance(); zup.advance(); f1z.advance();
    }
  }
  flush_counters(c, status);
}

// occupancy-derived persistent grid, cached per instantiation
template <class R, int RECON, int RS, int SM, int MINB> cudaError_t launch_ctu_fused(const SolveArgs<R>& a) {
  using C = CtuCfg<R, RECON, SM>;
  auto kern = ctu_fused_kernel<R, RECON, RS, SM, MINB>;
  const size_t smem = C::smem_bytes(a.g);
  if (smem > SMEM_MAX_OPTIN) return cudaErrorInvalidConfiguration;
  static int sms = 0;
  if (!sms) {
    int dev = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (sms <= 0) sms = 148;
  }
  cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  int per_sm = 0;
  e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, FNT, smem);
  if (e != cudaSuccess) return e;
  if (per_sm < 1) return cudaErrorInvalidConfiguration;
  long long grid = (long long)sms * per_sm;
  if (grid > a.Ng) grid = a.Ng;
  kern<<<(unsigned)grid, FNT, smem, a.stream>>>(a.in, a.out, a.face_flux, a.Ng, a.g, a.par, a.max_speed, a.cfl, a.status);
  return cudaGetLastError();
}

}  // namespace hydro
