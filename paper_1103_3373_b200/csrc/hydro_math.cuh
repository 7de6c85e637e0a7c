// hydro_math.cuh -- per-cell / per-face device arithmetic of the unsplit patch-group update.
//
// Schive, Zhang & Chiueh (arXiv:1103.3373).  The paper names the building blocks
// (PAPER.md:48 reconstruction + limiters, PAPER.md:39/46 characteristic tracing, PAPER.md:50
// Riemann solvers and the Roe fallback) and gives no formulas; the formulas are the readings
// listed in DESIGN.md ("Readings", S1-S24).  Everything here is templated on the arithmetic
// type R (float / double) and on compile-time direction / variant tags so that every 5-vector
// lives in registers (the paper's "5-element structs instead of arrays").
//
// This file is part of the CUDA product path.  It shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>

namespace hydro {

enum : int { SCHEME_MHM = 0, SCHEME_VL = 1, SCHEME_CTU = 2 };
enum : int { RS_EXACT = 0, RS_HLLE = 1, RS_HLLC = 2, RS_ROE = 3 };
enum : int { LIM_GMINMOD = 0, LIM_VANLEER = 1, LIM_VANALBADA = 2, LIM_HYBRID = 3 };
enum : int { RECON_PLM = 0, RECON_PPM = 1 };

constexpr int PS = 16;  // interior cells per side of a patch group

// ---- scalar helpers (one overload per precision) -------------------------------------------
__device__ __forceinline__ float  m_abs(float x) { return fabsf(x); }
__device__ __forceinline__ double m_abs(double x) { return fabs(x); }
__device__ __forceinline__ float  m_min(float a, float b) { return fminf(a, b); }
__device__ __forceinline__ double m_min(double a, double b) { return fmin(a, b); }
__device__ __forceinline__ float  m_max(float a, float b) { return fmaxf(a, b); }
__device__ __forceinline__ double m_max(double a, double b) { return fmax(a, b); }
__device__ __forceinline__ float  m_pow(float a, float b) { return powf(a, b); }
__device__ __forceinline__ double m_pow(double a, double b) { return pow(a, b); }

// Division / reciprocal / square-root policy.  fp64: IEEE-rounded.  fp32: the SFU approximations
// (div.approx / rcp.approx / sqrt.approx, <= 2 ulp, subnormals flushed), as the paper's own kernel did
// with -prec-div=false -ftz=true.  An IEEE fp32 division costs MUFU.RCP + FCHK + 4 FFMA +
// a branch to a slow-path subroutine, ~200 times per cell update; the error of the approximations is
// far inside the fp32 parity budget (L1 <= 1e-5 per step).  -DHYDRO_F32_IEEE=1
// restores IEEE fp32 arithmetic for A/B measurements.
#ifndef HYDRO_F32_IEEE
#define HYDRO_F32_IEEE 0
#endif
#if HYDRO_F32_IEEE
__device__ __forceinline__ float  m_sqrt(float x) { return sqrtf(x); }
__device__ __forceinline__ float  m_rcp(float x) { return 1.0f / x; }
__device__ __forceinline__ float  m_div(float a, float b) { return a / b; }
#else
__device__ __forceinline__ float  m_sqrt(float x) { float r; asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float  m_rcp(float x) { float r; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float  m_div(float a, float b) { float r; asm("div.approx.ftz.f32 %0, %1, %2;" : "=f"(r) : "f"(a), "f"(b)); return r; }
#endif
__device__ __forceinline__ double m_sqrt(double x) { return sqrt(x); }
__device__ __forceinline__ double m_rcp(double x) { return 1.0 / x; }
__device__ __forceinline__ double m_div(double a, double b) { return a / b; }

template <class R> struct ExactTol;
template <> struct ExactTol<float> { static __device__ __forceinline__ float v() { return 1e-6f; } };
template <> struct ExactTol<double> { static __device__ __forceinline__ double v() { return 1e-12; } };

template <class R> struct V5 {
  R q[5];
  __device__ __forceinline__ R& operator[](int i) { return q[i]; }
  __device__ __forceinline__ const R& operator[](int i) const { return q[i]; }
};

// IEEE bit patterns for the wave-speed maxima (hydro_dt, hydro_opts::next_max_speed): non-negative values order like
// their bits and the canonical NaN pattern is larger than +inf, so an integer atomicMax yields "max, or NaN if bad"
template <class R> struct Bits;
template <> struct Bits<float> {
  using U = unsigned int;
  static __device__ __forceinline__ U of(float x) { return __float_as_uint(x); }
  static __device__ __forceinline__ U nan() { return 0x7fc00000u; }
};
template <> struct Bits<double> {
  using U = unsigned long long;
  static __device__ __forceinline__ U of(double x) { return (U)__double_as_longlong(x); }
  static __device__ __forceinline__ U nan() { return 0x7ff8000000000000ull; }
};


// run-time parameters of one hydro_solve call (uniform over the grid)
template <class R> struct Par {
  R gamma, gm1;   // gamma, gamma-1
  R igm1;         // 1/(gamma-1), formed once on the host
  R ig1, ig2, sA0;  // 1/(gamma+1), 1/(2 gamma), sqrt(2/(gamma+1)): the exact solver's constants, formed once on the host
  R nu, hnu;      // dt/dh and half of it
  R theta;        // generalized-minmod coefficient (S7)
  R min_dens, min_pres;
  int limiter, char_limit, roe_fallback;
  R* next_speed;  // hydro_opts::next_max_speed (device scalar, zeroed by the host before the launch) or nullptr
  int next_norm;
};

// dt/dh from the device-resident hydro_dt result (hydro_opts::max_speed), uniform over the grid
template <class R> __device__ __forceinline__ void apply_device_dt(Par<R>& p, const R* max_speed, R cfl) {
  if (max_speed) {
    p.nu = m_div(cfl, __ldg(max_speed));
    p.hnu = R(0.5) * p.nu;
  }
}

// per-thread event counters, flushed to hydro_opts::status once per CTA
struct Cnt {
  int roe_fb;   // status[0]: Roe failures (fallback solver used)
  int bad;      // status[1]: non-positive rho / P seen by a conserved->primitive conversion
  int exact;    // status[2]: exact-solver vacuum / non-convergence
};

// ---- c0: conversions ------------------------------------------------------------------------
// U = (rho, mx, my, mz, E)  <->  W = (rho, vx, vy, vz, P),  E = P/(gamma-1) + rho |v|^2 / 2
template <class R> __device__ __forceinline__ V5<R> cons2prim(const V5<R>& U, const Par<R>& p, Cnt& c) {
  R rho = U[0];
  if (p.min_dens > R(0) && rho < p.min_dens) rho = p.min_dens;
  const R ir = m_rcp(rho);
  V5<R> W;
  W[0] = rho;
  W[1] = U[1] * ir;
  W[2] = U[2] * ir;
  W[3] = U[3] * ir;
  R P = p.gm1 * (U[4] - R(0.5) * rho * ((W[1] * W[1] + W[2] * W[2]) + W[3] * W[3]));
  if (!(U[0] > R(0)) || !(P > R(0))) c.bad++;
  if (p.min_pres > R(0) && P < p.min_pres) P = p.min_pres;
  W[4] = P;
  return W;
}
template <class R> __device__ __forceinline__ V5<R> prim2cons(const V5<R>& W, const Par<R>& p) {
  V5<R> U;
  U[0] = W[0];
  U[1] = W[0] * W[1];
  U[2] = W[0] * W[2];
  U[3] = W[0] * W[3];
  U[4] = W[4] * p.igm1 + R(0.5) * W[0] * ((W[1] * W[1] + W[2] * W[2]) + W[3] * W[3]);
  return U;
}

// normal-frame relabelling: (n, t1, t2) = (x,y,z), (y,z,x), (z,x,y) for D = 0,1,2
template <int D, class R> __device__ __forceinline__ V5<R> to_normal(const V5<R>& a) {
  V5<R> n;
  n[0] = a[0];
  n[1] = a[1 + D];
  n[2] = a[1 + (D + 1) % 3];
  n[3] = a[1 + (D + 2) % 3];
  n[4] = a[4];
  return n;
}
template <int D, class R> __device__ __forceinline__ V5<R> from_normal(const V5<R>& n) {
  V5<R> a;
  a[0] = n[0];
  a[1 + D] = n[1];
  a[1 + (D + 1) % 3] = n[2];
  a[1 + (D + 2) % 3] = n[3];
  a[4] = n[4];
  return a;
}

// physical flux and conserved vector of a normal-frame primitive state
template <class R> __device__ __forceinline__ void flux_and_cons(const V5<R>& W, const Par<R>& p, V5<R>& F, V5<R>& U) {
  const R rho = W[0], vn = W[1];
  const R E = W[4] * p.igm1 + R(0.5) * rho * ((vn * vn + W[2] * W[2]) + W[3] * W[3]);
  U[0] = rho;
  U[1] = rho * vn;
  U[2] = rho * W[2];
  U[3] = rho * W[3];
  U[4] = E;
  F[0] = U[1];
  F[1] = U[1] * vn + W[4];
  F[2] = U[1] * W[2];
  F[3] = U[1] * W[3];
  F[4] = (E + W[4]) * vn;
}
template <class R> __device__ __forceinline__ V5<R> phys_flux(const V5<R>& W, const Par<R>& p) {
  V5<R> F, U;
  flux_and_cons(W, p, F, U);
  return F;
}

// ---- c1: slope limiters ---------------------------------------------------------
template <class R> __device__ __forceinline__ R limited_slope(R dL, R dR, const Par<R>& p) {
  const R prod = dL * dR;
  if (!(prod > R(0))) return R(0);  // S19: zero product -> zero slope
  const R dC = R(0.5) * (dL + dR);
  switch (p.limiter) {
    case LIM_VANLEER: return m_div(R(2) * prod, dL + dR);
    case LIM_VANALBADA: return m_div(prod * (dL + dR), dL * dL + dR * dR);
    case LIM_GMINMOD: {
      const R m = m_min(m_min(p.theta * m_abs(dL), p.theta * m_abs(dR)), m_abs(dC));
      return dC > R(0) ? m : -m;
    }
    default: {  // hybrid: generalized minmod (theta = 2) combined with van Leer
      const R vl = m_abs(m_div(R(2) * prod, dL + dR));
      const R m = m_min(m_min(R(2) * m_abs(dL), R(2) * m_abs(dR)), m_min(m_abs(dC), vl));
      return dC > R(0) ? m : -m;
    }
  }
}

// eigen-system of the primitive normal-direction Jacobian at W (waves vn-c, vn, vn, vn, vn+c)
template <class R> struct Eig {
  R c, ic, ic2, rho, irho;
  __device__ __forceinline__ Eig(const V5<R>& W, const Par<R>& p) {
    rho = W[0];
    irho = m_rcp(rho);
    c = m_sqrt(p.gamma * W[4] * irho);
    ic = m_rcp(c);
    ic2 = ic * ic;
  }
  __device__ __forceinline__ V5<R> project(const V5<R>& d) const {  // a = L . d
    V5<R> a;
    const R x = d[4] * ic2, y = rho * d[1] * ic;
    a[0] = R(0.5) * (x - y);
    a[1] = d[0] - x;
    a[2] = d[2];
    a[3] = d[3];
    a[4] = R(0.5) * (x + y);
    return a;
  }
  __device__ __forceinline__ V5<R> expand(const V5<R>& a) const {  // sum_a a_a R_a
    V5<R> d;
    d[0] = (a[0] + a[1]) + a[4];
    d[1] = (c * irho) * (a[4] - a[0]);
    d[2] = a[2];
    d[3] = a[3];
    d[4] = (c * c) * (a[0] + a[4]);
    return d;
  }
};

// limited slope vector of the middle cell of (Wm, W0, Wp), normal-frame primitives
template <class R>
__device__ __forceinline__ V5<R> slope_vec(const V5<R>& Wm, const V5<R>& W0, const V5<R>& Wp, const Par<R>& p) {
  V5<R> dL, dR, s;
#pragma unroll
  for (int q = 0; q < 5; ++q) {
    dL[q] = W0[q] - Wm[q];
    dR[q] = Wp[q] - W0[q];
  }
  if (p.char_limit) {  // S8: limit the characteristic projections, then project back
    const Eig<R> e(W0, p);
    const V5<R> aL = e.project(dL), aR = e.project(dR);
    V5<R> a;
#pragma unroll
    for (int q = 0; q < 5; ++q) a[q] = limited_slope(aL[q], aR[q], p);
    return e.expand(a);
  }
#pragma unroll
  for (int q = 0; q < 5; ++q) s[q] = limited_slope(dL[q], dR[q], p);
  return s;
}

// ---- c2 + c3: face values of a cell from its normal-frame pencil ----------------------------
// PLM uses Wm1, W0, Wp1; PPM also Wm2, Wp2.  TRACE = CTU characteristic tracing to dt/2
// (PAPER.md:39, 46): reference-state form, approaching waves only (S5).
template <int RECON, bool TRACE, class R>
__device__ __forceinline__ void reconstruct(const V5<R>& Wm2, const V5<R>& Wm1, const V5<R>& W0, const V5<R>& Wp1,
                                            const V5<R>& Wp2, const Par<R>& p, V5<R>& Wlo, V5<R>& Wup) {
  const V5<R> dW = slope_vec(Wm1, W0, Wp1, p);
  V5<R> WL, WR, D, W6;
  if (RECON == RECON_PLM) {
#pragma unroll
    for (int q = 0; q < 5; ++q) {
      WL[q] = W0[q] - R(0.5) * dW[q];
      WR[q] = W0[q] + R(0.5) * dW[q];
    }
  } else {  // PPM: Colella-Woodward interpolation + monotonisation (S6)
    const V5<R> dWm = slope_vec(Wm2, Wm1, W0, p);
    const V5<R> dWp = slope_vec(W0, Wp1, Wp2, p);
#pragma unroll
    for (int q = 0; q < 5; ++q) {
      const R w0 = W0[q];
      R wl = R(0.5) * (Wm1[q] + w0) - (dW[q] - dWm[q]) * R(1.0 / 6.0);
      R wr = R(0.5) * (w0 + Wp1[q]) - (dWp[q] - dW[q]) * R(1.0 / 6.0);
      if ((wr - w0) * (w0 - wl) <= R(0)) {
        wl = w0;
        wr = w0;
      } else {
        const R dd = wr - wl, m6 = R(6) * (w0 - R(0.5) * (wl + wr));
        if (dd * m6 > dd * dd) wl = R(3) * w0 - R(2) * wr;
        else if (dd * m6 < -(dd * dd)) wr = R(3) * w0 - R(2) * wl;
      }
      WL[q] = wl;
      WR[q] = wr;
      D[q] = wr - wl;
      W6[q] = R(6) * (w0 - R(0.5) * (wl + wr));
    }
  }
  if (!TRACE) {
    Wlo = WL;
    Wup = WR;
    return;
  }
  const Eig<R> e(W0, p);
  const R vn = W0[1], lamM = vn + e.c, lam0 = vn - e.c, nu = p.nu;
  // wave speeds: index 0 -> vn-c, 1..3 -> vn, 4 -> vn+c
  if (RECON == RECON_PLM) {
    const V5<R> a = e.project(dW);
    V5<R> ap, am;
    // upper face: waves with lambda > 0, coefficient (nu/2)(lamM - lambda); the vn+c wave has coefficient 0
    const R cp0 = (lam0 > R(0)) ? R(0.5) * nu * (lamM - lam0) : R(0);
    const R cp1 = (vn > R(0)) ? R(0.5) * nu * (lamM - vn) : R(0);
    ap[0] = cp0 * a[0];
    ap[1] = cp1 * a[1];
    ap[2] = cp1 * a[2];
    ap[3] = cp1 * a[3];
    ap[4] = R(0);
    // lower face: waves with lambda < 0, coefficient (nu/2)(lam0 - lambda); the vn-c wave has coefficient 0
    const R cm1 = (vn < R(0)) ? R(0.5) * nu * (lam0 - vn) : R(0);
    const R cm4 = (lamM < R(0)) ? R(0.5) * nu * (lam0 - lamM) : R(0);
    am[0] = R(0);
    am[1] = cm1 * a[1];
    am[2] = cm1 * a[2];
    am[3] = cm1 * a[3];
    am[4] = cm4 * a[4];
    const V5<R> sp = e.expand(ap), sm = e.expand(am);
    const R fp = R(0.5) * nu * m_max(lamM, R(0)), fm = R(0.5) * nu * m_min(lam0, R(0));
#pragma unroll
    for (int q = 0; q < 5; ++q) {
      Wup[q] = (WR[q] - fp * dW[q]) + sp[q];
      Wlo[q] = (WL[q] - fm * dW[q]) + sm[q];
    }
  } else {
    const R sgp = nu * m_max(lamM, R(0)), sgm = nu * m_min(lam0, R(0));
    V5<R> DmW6, DpW6;
#pragma unroll
    for (int q = 0; q < 5; ++q) {
      DmW6[q] = D[q] - W6[q];
      DpW6[q] = D[q] + W6[q];
    }
    const V5<R> aDm = e.project(DmW6), aDp = e.project(DpW6), a6 = e.project(W6);
    const R n23 = nu * nu * R(1.0 / 3.0);
    // upper face (lambda > 0): A = (nu/2)(lamM - lambda), B = (nu^2/3)(lamM^2 - lambda^2)
    const bool p0 = lam0 > R(0), p1 = vn > R(0), m1 = vn < R(0), m4 = lamM < R(0);
    const R A0 = p0 ? R(0.5) * nu * (lamM - lam0) : R(0), B0 = p0 ? n23 * (lamM * lamM - lam0 * lam0) : R(0);
    const R A1 = p1 ? R(0.5) * nu * (lamM - vn) : R(0), B1 = p1 ? n23 * (lamM * lamM - vn * vn) : R(0);
    // lower face (lambda < 0): C = (nu/2)(lam0 - lambda), Dk = (nu^2/3)(lam0^2 - lambda^2)
    const R C1 = m1 ? R(0.5) * nu * (lam0 - vn) : R(0), D1 = m1 ? n23 * (lam0 * lam0 - vn * vn) : R(0);
    const R C4 = m4 ? R(0.5) * nu * (lam0 - lamM) : R(0), D4 = m4 ? n23 * (lam0 * lam0 - lamM * lamM) : R(0);
    V5<R> ap, am;
    ap[0] = A0 * aDm[0] + B0 * a6[0];
    ap[1] = A1 * aDm[1] + B1 * a6[1];
    ap[2] = A1 * aDm[2] + B1 * a6[2];
    ap[3] = A1 * aDm[3] + B1 * a6[3];
    ap[4] = R(0);
    am[0] = R(0);
    am[1] = C1 * aDp[1] + D1 * a6[1];
    am[2] = C1 * aDp[2] + D1 * a6[2];
    am[3] = C1 * aDp[3] + D1 * a6[3];
    am[4] = C4 * aDp[4] + D4 * a6[4];
    const V5<R> tp = e.expand(ap), tm = e.expand(am);
    const R kp = R(1) - R(2.0 / 3.0) * sgp, km = R(1) + R(2.0 / 3.0) * sgm;
#pragma unroll
    for (int q = 0; q < 5; ++q) {
      Wup[q] = (WR[q] - R(0.5) * sgp * (D[q] - kp * W6[q])) + tp[q];
      Wlo[q] = (WL[q] - R(0.5) * sgm * (D[q] + km * W6[q])) + tm[q];
    }
  }
}

// ---- c4: Riemann solvers in the normal frame ------------------------------------
template <class R> struct RoeAvg { R vn, v1, v2, H, a; };

template <class R>
__device__ __forceinline__ RoeAvg<R> roe_average(const V5<R>& WL, const V5<R>& WR, const V5<R>& UL, const V5<R>& UR,
                                                 const Par<R>& p) {
  const R HL = m_div(UL[4] + WL[4], WL[0]), HR = m_div(UR[4] + WR[4], WR[0]);
  const R sL = m_sqrt(WL[0]), sR = m_sqrt(WR[0]), id = m_rcp(sL + sR);
  RoeAvg<R> r;
  r.vn = (sL * WL[1] + sR * WR[1]) * id;
  r.v1 = (sL * WL[2] + sR * WR[2]) * id;
  r.v2 = (sL * WL[3] + sR * WR[3]) * id;
  r.H = (sL * HL + sR * HR) * id;
  const R q2 = (r.vn * r.vn + r.v1 * r.v1) + r.v2 * r.v2;
  r.a = m_sqrt(p.gm1 * (r.H - R(0.5) * q2));
  return r;
}

// HLLE (Einfeldt 1991): Roe-average and local signal speeds (S9)
template <class R>
__device__ __forceinline__ V5<R> hlle_from(const V5<R>& WL, const V5<R>& WR, const V5<R>& UL, const V5<R>& UR,
                                           const V5<R>& FL, const V5<R>& FR, const RoeAvg<R>& r, const Par<R>& p) {
  const R cL = m_sqrt(m_div(p.gamma * WL[4], WL[0])), cR = m_sqrt(m_div(p.gamma * WR[4], WR[0]));
  const R SL = m_min(r.vn - r.a, WL[1] - cL), SR = m_max(r.vn + r.a, WR[1] + cR);
  const R bm = m_min(SL, R(0)), bp = m_max(SR, R(0));
  const R iw = m_rcp(bp - bm), bb = bp * bm;
  V5<R> F;
#pragma unroll
  for (int q = 0; q < 5; ++q) F[q] = ((bp * FL[q] - bm * FR[q]) + bb * (UR[q] - UL[q])) * iw;
  return F;
}
template <class R> __device__ __forceinline__ V5<R> hlle(const V5<R>& WL, const V5<R>& WR, const Par<R>& p) {
  V5<R> UL, UR, FL, FR;
  flux_and_cons(WL, p, FL, UL);
  flux_and_cons(WR, p, FR, UR);
  const RoeAvg<R> r = roe_average(WL, WR, UL, UR, p);
  return hlle_from(WL, WR, UL, UR, FL, FR, r, p);
}

// HLLC with Toro's pressure-based wave-speed estimates (S9)
template <class R> __device__ __forceinline__ V5<R> hllc(const V5<R>& WL, const V5<R>& WR, const Par<R>& p) {
  const R g = p.gamma;
  const R cL = m_sqrt(m_div(g * WL[4], WL[0])), cR = m_sqrt(m_div(g * WR[4], WR[0]));
  const R rb = R(0.5) * (WL[0] + WR[0]), cb = R(0.5) * (cL + cR);
  const R ppv = R(0.5) * (WL[4] + WR[4]) - R(0.5) * (WR[1] - WL[1]) * rb * cb;
  const R ps = m_max(R(0), ppv);
  const R gf = m_div(g + R(1), R(2) * g);
  const R qL = (ps <= WL[4]) ? R(1) : m_sqrt(R(1) + gf * (m_div(ps, WL[4]) - R(1)));
  const R qR = (ps <= WR[4]) ? R(1) : m_sqrt(R(1) + gf * (m_div(ps, WR[4]) - R(1)));
  const R SL = WL[1] - cL * qL, SR = WR[1] + cR * qR;
  V5<R> UL, UR, FL, FR;
  flux_and_cons(WL, p, FL, UL);
  flux_and_cons(WR, p, FR, UR);
  if (SL >= R(0)) return FL;
  if (SR <= R(0)) return FR;
  const R mL = WL[0] * (SL - WL[1]), mR = WR[0] * (SR - WR[1]);
  const R Ss = m_div((WR[4] - WL[4]) + WL[1] * mL - WR[1] * mR, mL - mR);
  // pick the star region containing x/t = 0 (S19: S* = 0 -> left star)
  const bool left = Ss >= R(0);
  const V5<R>& WK = left ? WL : WR;
  const V5<R>& UK = left ? UL : UR;
  const V5<R>& FK = left ? FL : FR;
  const R SK = left ? SL : SR, mK = left ? mL : mR;
  const R f = m_div(mK, SK - Ss);
  V5<R> Us;
  Us[0] = f;
  Us[1] = f * Ss;
  Us[2] = f * WK[2];
  Us[3] = f * WK[3];
  Us[4] = f * (m_div(UK[4], WK[0]) + (Ss - WK[1]) * (Ss + m_div(WK[4], mK)));
  V5<R> F;
#pragma unroll
  for (int q = 0; q < 5; ++q) F[q] = FK[q] + SK * (Us[q] - UK[q]);
  return F;
}

// exact solver (Toro ch. 4; S11).  pressure function f_K(p) and its derivative
template <class R>
__device__ __forceinline__ void pressure_fn(R ps, R rhoK, R PK, R cK, const Par<R>& p, R& f, R& df) {
  const R g = p.gamma;
  if (ps > PK) {  // shock branch
    const R A = m_div(R(2), (g + R(1)) * rhoK), B = m_div(p.gm1, g + R(1)) * PK;
    const R s = m_sqrt(m_div(A, ps + B));
    f = (ps - PK) * s;
    df = s * (R(1) - m_div(ps - PK, R(2) * (B + ps)));
  } else {  // rarefaction branch
    const R pr = m_div(ps, PK);
    f = R(2) * cK * p.igm1 * (m_pow(pr, m_div(p.gm1, R(2) * g)) - R(1));
    df = m_div(m_pow(pr, m_div(-(g + R(1)), R(2) * g)), rhoK * cK);
  }
}

template <class R> __device__ __noinline__ V5<R> exact(const V5<R>& WL, const V5<R>& WR, const Par<R>& p, Cnt& c) {
  const R g = p.gamma;
  const R cL = m_sqrt(m_div(g * WL[4], WL[0])), cR = m_sqrt(m_div(g * WR[4], WR[0]));
  const R du = WR[1] - WL[1];
  if (R(2) * (cL + cR) * p.igm1 <= du) {  // vacuum generation -> HLLE flux
    c.exact++;
    return hlle(WL, WR, p);
  }
  const R epsp = R(1e-6) * m_min(WL[4], WR[4]);
  const R ppv = R(0.5) * (WL[4] + WR[4]) - R(0.125) * du * (WL[0] + WR[0]) * (cL + cR);
  R ps = m_max(epsp, ppv);
  R fL, dL, fR, dR;
  bool conv = false;
  for (int it = 0; it < 40; ++it) {
    pressure_fn(ps, WL[0], WL[4], cL, p, fL, dL);
    pressure_fn(ps, WR[0], WR[4], cR, p, fR, dR);
    R pn = ps - m_div((fL + fR) + du, dL + dR);
    if (!(pn > R(0))) pn = epsp;
    const R chg = m_div(R(2) * m_abs(pn - ps), pn + ps);
    ps = pn;
    if (chg < ExactTol<R>::v()) {
      conv = true;
      break;
    }
  }
  if (!conv) c.exact++;
  pressure_fn(ps, WL[0], WL[4], cL, p, fL, dL);
  pressure_fn(ps, WR[0], WR[4], cR, p, fR, dR);
  const R us = R(0.5) * (WL[1] + WR[1]) + R(0.5) * (fR - fL);
  // sample at x/t = 0 on the side of the contact given by sign(u*) (S19: u* = 0 -> left)
  const bool left = us >= R(0);
  const R sg = left ? R(1) : R(-1);  // mirror the right side onto the left-side formulas
  const R rK = left ? WL[0] : WR[0], PK = left ? WL[4] : WR[4], cK = left ? cL : cR;
  const R vK = left ? WL[1] : WR[1];
  const R mu = m_div(p.gm1, g + R(1));
  const R pr = m_div(ps, PK);
  V5<R> W;
  W[2] = left ? WL[2] : WR[2];
  W[3] = left ? WL[3] : WR[3];
  // in the mirrored frame velocities are s*v and the wave runs to the left
  if (ps > PK) {  // shock
    const R S = vK - sg * cK * m_sqrt(m_div(g + R(1), R(2) * g) * pr + m_div(p.gm1, R(2) * g));
    const bool undisturbed = left ? (S >= R(0)) : (S <= R(0));
    if (undisturbed) { W[0] = rK; W[1] = vK; W[4] = PK; }
    else { W[0] = m_div(rK * (pr + mu), mu * pr + R(1)); W[1] = us; W[4] = ps; }
  } else {  // rarefaction
    const R head = vK - sg * cK;
    const R cs = cK * m_pow(pr, m_div(p.gm1, R(2) * g));
    const R tail = us - sg * cs;
    const bool before_head = left ? (head >= R(0)) : (head <= R(0));
    const bool behind_tail = left ? (tail <= R(0)) : (tail >= R(0));
    if (before_head) { W[0] = rK; W[1] = vK; W[4] = PK; }
    else if (behind_tail) { W[0] = rK * m_pow(pr, m_rcp(g)); W[1] = us; W[4] = ps; }
    else {
      const R phi = m_div(R(2), g + R(1)) + m_div(sg * mu * vK, cK);
      W[0] = rK * m_pow(phi, R(2) * p.igm1);
      W[1] = m_div(R(2), g + R(1)) * (sg * cK + R(0.5) * p.gm1 * vK);
      W[4] = PK * m_pow(phi, R(2) * g * p.igm1);
    }
  }
  return phys_flux(W, p);
}

// Roe's solver (Roe 1981), no entropy fix; Athena-style failure test + fallback
template <class R> __device__ __forceinline__ V5<R> roe(const V5<R>& WL, const V5<R>& WR, const Par<R>& p, Cnt& c) {
  V5<R> UL, UR, FL, FR;
  flux_and_cons(WL, p, FL, UL);
  flux_and_cons(WR, p, FR, UR);
  const RoeAvg<R> r = roe_average(WL, WR, UL, UR, p);
  const R vn = r.vn, v1 = r.v1, v2 = r.v2, H = r.H, a = r.a;
  const R q2 = (vn * vn + v1 * v1) + v2 * v2;
  V5<R> du;
#pragma unroll
  for (int q = 0; q < 5; ++q) du[q] = UR[q] - UL[q];
  const R a3 = du[2] - v1 * du[0], a4 = du[3] - v2 * du[0];
  const R du5 = (du[4] - a3 * v1) - a4 * v2;
  const R ia = m_rcp(a);
  const R a2 = p.gm1 * (ia * ia) * ((du[0] * (H - vn * vn) + vn * du[1]) - du5);
  const R a1 = ((du[0] * (vn + a) - du[1]) - a * a2) * (R(0.5) * ia);
  const R a5 = du[0] - (a1 + a2);
  const R K1[5] = {R(1), vn - a, v1, v2, H - vn * a};
  const R K2[5] = {R(1), vn, v1, v2, R(0.5) * q2};
  const R K5[5] = {R(1), vn + a, v1, v2, H + vn * a};
  // failure test on the two intermediate states U_L + a1 K1 and U_R - a5 K5
  R A[5], B[5];
#pragma unroll
  for (int q = 0; q < 5; ++q) {
    A[q] = UL[q] + a1 * K1[q];
    B[q] = UR[q] - a5 * K5[q];
  }
  const R PA = p.gm1 * (A[4] - R(0.5) * m_div((A[1] * A[1] + A[2] * A[2]) + A[3] * A[3], A[0]));
  const R PB = p.gm1 * (B[4] - R(0.5) * m_div((B[1] * B[1] + B[2] * B[2]) + B[3] * B[3], B[0]));
  if (!(A[0] > R(0)) || !(PA > R(0)) || !(B[0] > R(0)) || !(PB > R(0))) {
    c.roe_fb++;
    if (p.roe_fallback == 2) return hllc(WL, WR, p);
    if (p.roe_fallback == 3) return exact(WL, WR, p, c);
    return hlle_from(WL, WR, UL, UR, FL, FR, r, p);
  }
  const R l1 = m_abs(vn - a), l2 = m_abs(vn), l5 = m_abs(vn + a);
  const R w1 = a1 * l1, w2 = a2 * l2, w3 = a3 * l2, w4 = a4 * l2, w5 = a5 * l5;
  V5<R> F;
  // K3 = (0,0,1,0,v1), K4 = (0,0,0,1,v2)
  const R d0 = (w1 + w2) + w5;
  const R d1 = (w1 * K1[1] + w2 * K2[1]) + w5 * K5[1];
  const R d2 = ((w1 * v1 + w2 * v1) + w3) + w5 * v1;
  const R d3 = (((w1 * v2 + w2 * v2)) + w4) + w5 * v2;
  const R d4 = (((w1 * K1[4] + w2 * K2[4]) + w3 * v1) + w4 * v2) + w5 * K5[4];
  F[0] = R(0.5) * (FL[0] + FR[0]) - R(0.5) * d0;
  F[1] = R(0.5) * (FL[1] + FR[1]) - R(0.5) * d1;
  F[2] = R(0.5) * (FL[2] + FR[2]) - R(0.5) * d2;
  F[3] = R(0.5) * (FL[3] + FR[3]) - R(0.5) * d3;
  F[4] = R(0.5) * (FL[4] + FR[4]) - R(0.5) * d4;
  return F;
}

// dispatch on the compile-time solver tag; inputs/outputs in the normal frame
template <int RS, class R>
__device__ __forceinline__ V5<R> riemann_n(const V5<R>& WL, const V5<R>& WR, const Par<R>& p, Cnt& c) {
  if (RS == RS_EXACT) return exact(WL, WR, p, c);
  if (RS == RS_HLLE) return hlle(WL, WR, p);
  if (RS == RS_HLLC) return hllc(WL, WR, p);
  return roe(WL, WR, p, c);
}
// xyz-frame wrapper: face normal D, states and flux in (rho, x, y, z, P/E) order
template <int RS, int D, class R>
__device__ __forceinline__ V5<R> riemann_d(const V5<R>& WL, const V5<R>& WR, const Par<R>& p, Cnt& c) {
  return from_normal<D>(riemann_n<RS>(to_normal<D>(WL), to_normal<D>(WR), p, c));
}

// add the per-thread event counters of a CTA to hydro_opts::status
__device__ __forceinline__ void flush_counters(const Cnt& c, long long* status) {
  if (!status) return;
  // warp-aggregate, then one atomic per warp and counter (rare events; status may be nullptr)
  int v[3] = {c.roe_fb, c.bad, c.exact};
#pragma unroll
  for (int q = 0; q < 3; ++q) {
    int s = v[q];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if ((threadIdx.x & 31) == 0 && s) atomicAdd(reinterpret_cast<unsigned long long*>(status + q), (unsigned long long)s);
  }
}

}  // namespace hydro
