// hydro_lean_math.cuh -- instruction-lean forms of the per-cell / per-face arithmetic for the
// dominant variants (PLM + van Leer limiter on primitive variables, no floors; Roe and HLLC solvers).
//
// Same readings as hydro_math.cuh (S1-S24), algebraically rearranged so that the kernel
// issues fewer instructions: the profile of the first fused kernels showed the path bound by
// instruction issue, not by HBM (profiles/r1_ncu_fused_f32_v1.md), so what counts is the number of
// FP32/FP64 + MUFU instructions per Riemann solve and per reconstruction.
//   * branch-free limiter and tracing (selects, no divergent control flow);
//   * the characteristic projection of the tracing written out per component with one rsqrt
//     (1/(rho c)) instead of rcp + sqrt + rcp;
//   * Roe wave strengths from the primitive jumps (drho, du, dp with rho~ = sqrt(rhoL rhoR)), which
//     equal the conserved-jump strengths of S-c4 identically for Roe averages (Roe 1981, sec. 4);
//     enthalpy from H = gamma/(gamma-1) P/rho + |v|^2/2 and the energy flux as (rho u) H;
//   * the Roe failure test without divisions: P* > 0  <=>  2 E* rho* - |m*|^2 > 0.
// Results differ from hydro_math.cuh by rounding only; parity with the oracle is what tests/ checks.
// Part of the CUDA product path; shares nothing with oracle/.
#pragma once
#include "hydro_math.cuh"

namespace hydro {

#if HYDRO_F32_IEEE
__device__ __forceinline__ float m_rsqrt(float x) { return 1.0f / sqrtf(x); }
#else
__device__ __forceinline__ float m_rsqrt(float x) { float r; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
#endif
__device__ __forceinline__ double m_rsqrt(double x) { return rsqrt(x); }  // <= 1 ulp, no division
__device__ __forceinline__ float m_fma(float a, float b, float c) { return fmaf(a, b, c); }
__device__ __forceinline__ double m_fma(double a, double b, double c) { return fma(a, b, c); }

// Division-like operations of the lean path.  fp32: the SFU approximations of hydro_math.cuh.  fp64: an IEEE division
// or square root is ~20 instructions with a branch to a slow path; the lean path instead refines the SFU's
// 2^-23 seed (rcp.approx.ftz.f64 / rsqrt.approx.ftz.f64) with one third-order step in FMAs: branch-free, <= 2 ulp,
// far inside the fp64 parity budget.  Zero / denormal arguments give inf / NaN, which every
// caller either discards by a select (limiter) or routes to the Roe failure test; -DHYDRO_F64_IEEE=1 restores
// IEEE operations for A/B measurements.
#ifndef HYDRO_F64_IEEE
#define HYDRO_F64_IEEE 0
#endif
#ifndef LEAN_EXACT_SELECT
#define LEAN_EXACT_SELECT 1
#endif
#ifndef LEAN_DIV_REFINE
#define LEAN_DIV_REFINE 0
#endif
__device__ __forceinline__ float l_rcp(float x) { return m_rcp(x); }
__device__ __forceinline__ float l_div(float a, float b) { return m_div(a, b); }
__device__ __forceinline__ float l_sqrt(float x) { return m_sqrt(x); }
__device__ __forceinline__ float l_rsqrt(float x) { return m_rsqrt(x); }
#if HYDRO_F64_IEEE
__device__ __forceinline__ double l_rcp(double x) { return 1.0 / x; }
__device__ __forceinline__ double l_div(double a, double b) { return a / b; }
__device__ __forceinline__ double l_sqrt(double x) { return sqrt(x); }
__device__ __forceinline__ double l_rsqrt(double x) { return rsqrt(x); }
#else
// one THIRD-order step from the 2^-23 seed (error e^3 ~ 2^-69, then the rounding of the last two operations): three / five
// FP64-pipe instructions instead of the four / eight of two Newton steps -- the FP64 pipe (two issue cycles per warp
// instruction) is what bounds the fp64 kernels
__device__ __forceinline__ double l_rcp(double x) {
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
  const double e = fma(-x, r, 1.0);          // 1 - x r
  return fma(r, fma(e, e, e), r);            // r (1 + e + e^2)
}
#if LEAN_DIV_REFINE
__device__ __forceinline__ double l_div(double a, double b) {
  const double r = l_rcp(b), q = a * r;
  return fma(fma(-b, q, a), r, q);
}
#else
__device__ __forceinline__ double l_div(double a, double b) { return a * l_rcp(b); }  // <= 1.5 ulp; the residual step cost two more FP64-pipe instructions
#endif
__device__ __forceinline__ double l_rsqrt(double x) {
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  const double e = fma(-x * y, y, 1.0);      // 1 - x y^2
  return fma(y, fma(0.375, e, 0.5) * e, y);  // y (1 + e/2 + 3 e^2 / 8)
}
__device__ __forceinline__ double l_sqrt(double x) {
  const double y = l_rsqrt(x), s = x * y;
  return fma(fma(-s, s, x), 0.5 * y, s);
}
#endif

// ---- c0: conversions --------------------------------------------------------------------------
// non-positive rho / P seen by a conversion (status[1]).  `int&`: one count per conversion.  `BadMin&` (the fp32 CTU kernel,
// which is bound by instruction issue): a NaN-propagating running minimum of every rho and P converted -- one FMNMX3.NAN
// instead of two compares and an add -- tested and reset once per plane step, so there status[1] counts (thread, step)
// pairs that met a bad state: non-zero exactly when the per-conversion count is.
struct BadMin { float mn; };
__device__ __forceinline__ void note_state(int& bad, float rho, float P) { bad += (rho > 0.f && P > 0.f) ? 0 : 1; }
__device__ __forceinline__ void note_state(int& bad, double rho, double P) { bad += (rho > 0.0 && P > 0.0) ? 0 : 1; }
__device__ __forceinline__ void note_state(BadMin& b, float rho, float P) {
  asm("min.NaN.f32 %0, %0, %1, %2;" : "+f"(b.mn) : "f"(rho), "f"(P));
}
template <class R> struct BadTrk { using type = int; };
template <> struct BadTrk<float> { using type = BadMin; };
__device__ __forceinline__ void trk_reset(int& t) { t = 0; }
__device__ __forceinline__ void trk_reset(BadMin& t) { t.mn = 1.0f; }
__device__ __forceinline__ int trk_flush(int& t) { const int n = t; t = 0; return n; }
__device__ __forceinline__ int trk_flush(BadMin& t) { const int n = (t.mn > 0.0f) ? 0 : 1; t.mn = 1.0f; return n; }

// rho |v|^2 is formed as m . v (3 instructions)
template <class R, class T> __device__ __forceinline__ V5<R> lean_cons2prim(const V5<R>& U, const Par<R>& p, T& bad) {
  const R ir = l_rcp(U[0]);
  V5<R> W;
  W[0] = U[0];
  W[1] = U[1] * ir;
  W[2] = U[2] * ir;
  W[3] = U[3] * ir;
  const R mv = m_fma(U[3], W[3], m_fma(U[2], W[2], U[1] * W[1]));
  W[4] = p.gm1 * m_fma(R(-0.5), mv, U[4]);
  note_state(bad, U[0], W[4]);
  return W;
}

// transverse correction of one face state: W <- prim(cons(W) - dq)
template <class R, class T> __device__ __forceinline__ V5<R> lean_correct(const V5<R>& W, const V5<R>& dq, const Par<R>& p, T& bad) {
  V5<R> U;
  U[0] = W[0] - dq[0];
  U[1] = m_fma(W[0], W[1], -dq[1]);
  U[2] = m_fma(W[0], W[2], -dq[2]);
  U[3] = m_fma(W[0], W[3], -dq[3]);
  const R q2 = m_fma(W[3], W[3], m_fma(W[2], W[2], W[1] * W[1]));
  U[4] = m_fma(W[4], p.igm1, m_fma(R(0.5) * W[0], q2, -dq[4]));
  return lean_cons2prim(U, p, bad);
}

// ---- c6 fused into the update: wave speed of the UPDATED cell for the next step's dt (hydro_opts::next_max_speed)
template <class R> __device__ __forceinline__ void track_speed(const V5<R>& W, const Par<R>& p, typename Bits<R>::U& best) {
  using U = typename Bits<R>::U;
  const R c = l_sqrt(p.gamma * W[4] * l_rcp(W[0]));
  const R ax = m_abs(W[1]), ay = m_abs(W[2]), az = m_abs(W[3]);
  const R s = p.next_norm == 0 ? m_max(m_max(ax, ay), az) + c : ((ax + ay) + az) + R(3) * c;
  const bool bad = !(W[0] > R(0)) || !(W[4] > R(0)) || !(s == s);
  const U bits = bad ? Bits<R>::nan() : Bits<R>::of(s);
  best = bits > best ? bits : best;
}
template <class R> __device__ __forceinline__ void flush_speed(typename Bits<R>::U best, R* dst) {
  using U = typename Bits<R>::U;
  if (!dst) return;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    const U other = __shfl_xor_sync(0xffffffffu, best, o);
    best = other > best ? other : best;
  }
  if ((threadIdx.x & 31) == 0 && best) atomicMax(reinterpret_cast<U*>(dst), best);
}

// ---- c1-c3: PLM + van Leer limiter on primitive variables + CTU tracing (normal frame) ---------
template <class R> __device__ __forceinline__ R vl_slope(R dL, R dR) {
  const R prod = dL * dR;
  const R s = l_div(prod + prod, dL + dR);
  return prod > R(0) ? s : R(0);  // S19; the select also discards inf/NaN of the unused quotient
}
// HALF the van Leer slope, dL dR / (dL + dR): the factor 2 moves into the (compile-time or per-cell) coefficients that
// multiply the slope, which is exact in binary arithmetic -- results are bitwise those of vl_slope, with one add less per slope
template <class R> __device__ __forceinline__ R vl_half_slope(R dL, R dR) {
  const R prod = dL * dR;
  const R s = l_div(prod, dL + dR);
  return prod > R(0) ? s : R(0);
}

template <class R>
__device__ __forceinline__ void lean_plm_trace(const V5<R>& Wm, const V5<R>& W0, const V5<R>& Wp, const Par<R>& p, R nu, R hnu,
                                               V5<R>& lo, V5<R>& up) {
  V5<R> s;  // HALF slopes (vl_half_slope); every coefficient below carries the factor 2
#pragma unroll
  for (int q = 0; q < 5; ++q) s[q] = vl_half_slope(W0[q] - Wm[q], Wp[q] - W0[q]);
  // eigen-system scalars from one rsqrt: irc = 1/(rho c), c = gamma P irc, 1/c = rho irc
  const R gP = p.gamma * W0[4], x = gP * W0[0];
  const R irc = l_rsqrt(x);
  const R c = gP * irc, ic = W0[0] * irc, ic2 = ic * ic, rc = x * irc;
  const R u = W0[1], lamM = u + c, lam0 = u - c;
  const R nc = nu * c;
  // S5 / S19: only waves approaching the face, lambda = 0 contributes to neither
  const R b0 = lam0 > R(0) ? nc : R(0);     // (nu/2)(lamM - lam0), applied to a FULL amplitude below
  const R b1 = u > R(0) ? nc : R(0);        // 2 (nu/2)(lamM - u)
  const R g1 = u < R(0) ? -nc : R(0);       // 2 (nu/2)(lam0 - u)
  const R g4 = lamM < R(0) ? -nc : R(0);    // (nu/2)(lam0 - lamM)
  const R kp = m_fma(-nu, m_max(lamM, R(0)), R(1));   // 2 (1/2 - (nu/2) max(lamM, 0))
  const R km = m_fma(-nu, m_min(lam0, R(0)), R(-1));
  const R Z = rc * s[1];                          // rho c du / 2
  const R B0 = b0 * (s[4] - Z);                   // coefficient x (L_0 . s) c^2: half slopes give (dP - rho c du) / 2 directly
  const R B4 = g4 * (s[4] + Z);
  const R e1 = m_fma(-s[4], ic2, s[0]);           // half the entropy-wave amplitude
  up[0] = m_fma(B0, ic2, m_fma(b1, e1, m_fma(kp, s[0], W0[0])));
  up[1] = m_fma(-B0, irc, m_fma(kp, s[1], W0[1]));
  up[2] = m_fma(kp + b1, s[2], W0[2]);
  up[3] = m_fma(kp + b1, s[3], W0[3]);
  up[4] = m_fma(kp, s[4], W0[4]) + B0;
  lo[0] = m_fma(B4, ic2, m_fma(g1, e1, m_fma(km, s[0], W0[0])));
  lo[1] = m_fma(B4, irc, m_fma(km, s[1], W0[1]));
  lo[2] = m_fma(km + g1, s[2], W0[2]);
  lo[3] = m_fma(km + g1, s[3], W0[3]);
  lo[4] = m_fma(km, s[4], W0[4]) + B4;
}

// ---- c2-c3: PPM (S6: Colella-Woodward interpolation + monotonisation, no steepening / flattening), van Leer slopes on
// primitive variables, branch-free.  Parabola of the middle cell: edge values wl, wr; D = wr - wl; W6 = 6 (w0 - (wl+wr)/2)
template <class R>
__device__ __forceinline__ void lean_ppm_parabola(const V5<R>& Wm2, const V5<R>& Wm1, const V5<R>& W0, const V5<R>& Wp1,
                                                  const V5<R>& Wp2, V5<R>& WL, V5<R>& WR) {
#pragma unroll
  for (int q = 0; q < 5; ++q) {
    const R w0 = W0[q];
    const R dLm = Wm1[q] - Wm2[q], dL = w0 - Wm1[q], dR = Wp1[q] - w0, dRp = Wp2[q] - Wp1[q];
    const R sm = vl_half_slope(dLm, dL), s0 = vl_half_slope(dL, dR), sp = vl_half_slope(dR, dRp);  // half slopes: -1/6 -> -1/3
    R wl = m_fma(R(-1.0 / 3.0), s0 - sm, R(0.5) * (Wm1[q] + w0));
    R wr = m_fma(R(-1.0 / 3.0), sp - s0, R(0.5) * (w0 + Wp1[q]));
    const bool ext = (wr - w0) * (w0 - wl) <= R(0);
    const R dd = wr - wl, m6 = R(6) * m_fma(R(-0.5), wl + wr, w0);
    const R t = dd * m6, d2 = dd * dd;
    const bool c1 = t > d2, c2 = !c1 && t < -d2;
    const R wl1 = m_fma(R(-2), wr, R(3) * w0), wr1 = m_fma(R(-2), wl, R(3) * w0);
    wl = ext ? w0 : (c1 ? wl1 : wl);
    wr = ext ? w0 : (c2 ? wr1 : wr);
    WL[q] = wl;
    WR[q] = wr;
  }
}
// untraced PPM face values (MHM, VL)
template <class R>
__device__ __forceinline__ void lean_ppm(const V5<R>& Wm2, const V5<R>& Wm1, const V5<R>& W0, const V5<R>& Wp1, const V5<R>& Wp2,
                                         V5<R>& lo, V5<R>& up) {
  lean_ppm_parabola(Wm2, Wm1, W0, Wp1, Wp2, lo, up);
}
// PPM + CTU characteristic tracing to dt/2 (S5: reference-state form, approaching waves only), normal frame
template <class R>
__device__ __forceinline__ void lean_ppm_trace(const V5<R>& Wm2, const V5<R>& Wm1, const V5<R>& W0, const V5<R>& Wp1,
                                               const V5<R>& Wp2, const Par<R>& p, R nu, V5<R>& lo, V5<R>& up) {
  V5<R> WL, WR, D, W6;
  lean_ppm_parabola(Wm2, Wm1, W0, Wp1, Wp2, WL, WR);
#pragma unroll
  for (int q = 0; q < 5; ++q) {
    D[q] = WR[q] - WL[q];
    W6[q] = R(6) * m_fma(R(-0.5), WL[q] + WR[q], W0[q]);
  }
  const R gP = p.gamma * W0[4], x = gP * W0[0];
  const R irc = l_rsqrt(x);
  const R c = gP * irc, ic = W0[0] * irc, ic2 = ic * ic, rc = x * irc;
  const R u = W0[1], lamM = u + c, lam0 = u - c;
  const R nc = nu * c, n23 = nu * nu * R(1.0 / 3.0), uc = u * c, c2 = c * c;
  // upper face (lambda > 0): A = (nu/2)(lamM - lambda), B = (nu^2/3)(lamM^2 - lambda^2); per wave V = A D + (B - A) W6
  const bool p0 = lam0 > R(0), p1 = u > R(0), m1 = u < R(0), m4 = lamM < R(0);
  const R A0 = p0 ? nc : R(0), BA0 = p0 ? m_fma(n23, R(4) * uc, -nc) : R(0);
  const R A1 = p1 ? R(0.5) * nc : R(0), BA1 = p1 ? m_fma(n23, uc + uc + c2, R(-0.5) * nc) : R(0);
  // lower face (lambda < 0): C = (nu/2)(lam0 - lambda), Dk = (nu^2/3)(lam0^2 - lambda^2); per wave V = C D + (C + Dk) W6
  const R C1 = m1 ? R(-0.5) * nc : R(0), CD1 = m1 ? m_fma(n23, c2 - (uc + uc), R(-0.5) * nc) : R(0);
  const R C4 = m4 ? -nc : R(0), CD4 = m4 ? m_fma(n23, R(-4) * uc, -nc) : R(0);
  const R sgp = nu * m_max(lamM, R(0)), sgm = nu * m_min(lam0, R(0));
  const R kp = m_fma(R(-2.0 / 3.0), sgp, R(1)), km = m_fma(R(2.0 / 3.0), sgm, R(1));
  const R hp = R(-0.5) * sgp, hm = R(-0.5) * sgm;
  // acoustic amplitudes times c^2: (L . V) c^2 = (V_P -+ rho c V_u) / 2
  const R V0u = m_fma(A0, D[1], BA0 * W6[1]), V0p = m_fma(A0, D[4], BA0 * W6[4]);
  const R V4u = m_fma(C4, D[1], CD4 * W6[1]), V4p = m_fma(C4, D[4], CD4 * W6[4]);
  const R B0 = R(0.5) * m_fma(-rc, V0u, V0p), B4 = R(0.5) * m_fma(rc, V4u, V4p);
  // entropy / shear waves
  V5<R> V1, Vm;
#pragma unroll
  for (int q = 0; q < 5; ++q) {
    V1[q] = m_fma(A1, D[q], BA1 * W6[q]);
    Vm[q] = m_fma(C1, D[q], CD1 * W6[q]);
  }
  V5<R> bu, bl;  // W_R - (sgp/2)(D - kp W6),  W_L - (sgm/2)(D + km W6)
#pragma unroll
  for (int q = 0; q < 5; ++q) {
    bu[q] = m_fma(hp, m_fma(-kp, W6[q], D[q]), WR[q]);
    bl[q] = m_fma(hm, m_fma(km, W6[q], D[q]), WL[q]);
  }
  up[0] = m_fma(B0, ic2, m_fma(-V1[4], ic2, V1[0])) + bu[0];
  up[1] = m_fma(-B0, irc, bu[1]);
  up[2] = bu[2] + V1[2];
  up[3] = bu[3] + V1[3];
  up[4] = bu[4] + B0;
  lo[0] = m_fma(B4, ic2, m_fma(-Vm[4], ic2, Vm[0])) + bl[0];
  lo[1] = m_fma(B4, irc, bl[1]);
  lo[2] = bl[2] + Vm[2];
  lo[3] = bl[3] + Vm[3];
  lo[4] = bl[4] + B4;
}

// ---- c4: Roe's solver, primitive-jump form (normal frame in, normal-frame flux out) ------------
// per-state quantities of a Riemann problem
template <class R> struct LeanState { R ir, sq, H, m, F1; };  // the other flux components are m v, m w, m H
template <class R> __device__ __forceinline__ LeanState<R> lean_state(const V5<R>& W, R g1) {
  LeanState<R> s;
  if (sizeof(R) == 4) {  // fp32: two SFU instructions are cheaper than the extra multiplies
    s.ir = l_rcp(W[0]);
    s.sq = l_sqrt(W[0]);
  } else {               // fp64: one rsqrt instead of a division and a square root
    const R is = l_rsqrt(W[0]);
    s.ir = is * is;
    s.sq = W[0] * is;
  }
  const R q2 = m_fma(W[3], W[3], m_fma(W[2], W[2], W[1] * W[1]));
  s.H = m_fma(R(0.5), q2, (g1 * W[4]) * s.ir);
  s.m = W[0] * W[1];
  s.F1 = m_fma(s.m, W[1], W[4]);
  return s;
}

// the rare path: Roe failed at this face -> HLLE / HLLC / exact flux of the same states.  Everything
// crosses the call by value (registers): a pointer argument would put the caller's states AND its flux on the stack
// in the hot path (23.5 M local stores per launch in the round-1 kernel).
template <class R> struct FluxRet { R f0, f1, f2, f3, f4; int ex; };
template <class R>
__device__ __noinline__ FluxRet<R> roe_fallback_flux(R l0, R l1, R l2, R l3, R l4, R r0, R r1, R r2, R r3, R r4, R gamma, R gm1,
                                                     R igm1, int mode) {
  Par<R> p;
  p.gamma = gamma; p.gm1 = gm1; p.igm1 = igm1; p.roe_fallback = mode;
  p.ig1 = p.ig2 = p.sA0 = R(0);  // the generic solvers of hydro_math.cuh form their own constants
  p.nu = p.hnu = p.theta = p.min_dens = p.min_pres = R(0);
  p.limiter = p.char_limit = p.next_norm = 0;
  p.next_speed = nullptr;
  V5<R> WL, WR, F;
  WL[0] = l0; WL[1] = l1; WL[2] = l2; WL[3] = l3; WL[4] = l4;
  WR[0] = r0; WR[1] = r1; WR[2] = r2; WR[3] = r3; WR[4] = r4;
  Cnt c = {0, 0, 0};
  if (mode == 2) F = hllc(WL, WR, p);
  else if (mode == 3) F = exact(WL, WR, p, c);
  else F = hlle(WL, WR, p);
  FluxRet<R> r = {F[0], F[1], F[2], F[3], F[4], c.exact};
  return r;
}

// fp64: thirteen doubles by value are 26 argument registers at every call site; there the two states cross by pointer (copied
// to the stack inside the cold branch only) and just the flux comes back by value
template <class R>
__device__ __noinline__ FluxRet<R> roe_fallback_flux_p(const V5<R>* WL, const V5<R>* WR, R gamma, R gm1, R igm1, int mode) {
  return roe_fallback_flux<R>((*WL)[0], (*WL)[1], (*WL)[2], (*WL)[3], (*WL)[4], (*WR)[0], (*WR)[1], (*WR)[2], (*WR)[3], (*WR)[4],
                              gamma, gm1, igm1, mode);
}

// branch-free core: the Roe flux and whether both intermediate states passed the failure test.  Keeping the
// (rare) fallback out of it lets two independent solves share one basic block and interleave.
// hs: the flux is returned times 2 hs (0.5: the flux itself; the CTU first pass asks for nu/2 times the flux at no extra cost)
template <class R> __device__ __forceinline__ bool lean_roe_core(const V5<R>& WL, const V5<R>& WR, const Par<R>& p, V5<R>& F, R hs = R(0.5)) {
  const R g1 = p.gamma * p.igm1;
  const LeanState<R> L = lean_state(WL, g1), Rr = lean_state(WR, g1);
  // Roe averages with weights wL = sqrt(rhoL)/(sqrt(rhoL)+sqrt(rhoR)), wR = 1 - wL; rho~ = sqrt(rhoL rhoR)
  const R wR = Rr.sq * l_rcp(L.sq + Rr.sq);
  const R rt = L.sq * Rr.sq;
  const R du = WR[1] - WL[1], dv = WR[2] - WL[2], dw = WR[3] - WL[3];
  const R ut = m_fma(wR, du, WL[1]), vt = m_fma(wR, dv, WL[2]), wt = m_fma(wR, dw, WL[3]);
  const R Ht = m_fma(wR, Rr.H - L.H, L.H);
  const R hq = R(0.5) * m_fma(wt, wt, m_fma(vt, vt, ut * ut));
  const R a2 = p.gm1 * (Ht - hq);
  R a, ia2;
  if (sizeof(R) == 4) { a = l_sqrt(a2); ia2 = l_rcp(a2); }
  else { const R ia = l_rsqrt(a2); a = a2 * ia; ia2 = ia * ia; }
  // wave strengths from the primitive jumps
  const R dp = WR[4] - WL[4], dr = WR[0] - WL[0];
  const R y = (rt * a) * du, h = R(0.5) * ia2;
  const R al1 = (dp - y) * h, al5 = (dp + y) * h, al2 = m_fma(-dp, ia2, dr);
  const R al3 = rt * dv, al4 = rt * dw;
  const R um = ut - a, up = ut + a, ua = ut * a, H1 = Ht - ua, H5 = Ht + ua;
  // failure test on U_L + al1 K1 and U_R - al5 K5 (rho > 0 and P > 0, the latter without a division)
  const R A0 = WL[0] + al1, B0 = WR[0] - al5;
  const R A1 = m_fma(al1, um, L.m), B1 = m_fma(-al5, up, Rr.m);
  const R A2 = m_fma(al1, vt, WL[0] * WL[2]), B2 = m_fma(-al5, vt, WR[0] * WR[2]);
  const R A3 = m_fma(al1, wt, WL[0] * WL[3]), B3 = m_fma(-al5, wt, WR[0] * WR[3]);
  const R A4 = m_fma(al1, H1, m_fma(WL[0], L.H, -WL[4])), B4 = m_fma(-al5, H5, m_fma(WR[0], Rr.H, -WR[4]));
  const R mA = m_fma(A3, A3, m_fma(A2, A2, A1 * A1)), mB = m_fma(B3, B3, m_fma(B2, B2, B1 * B1));
  const R tA = m_fma(A4 + A4, A0, -mA), tB = m_fma(B4 + B4, B0, -mB);
  const bool ok = A0 > R(0) && B0 > R(0) && tA > R(0) && tB > R(0);  // NaN fails the test
  const R w1 = al1 * m_abs(um), w2 = al2 * m_abs(ut), w5 = al5 * m_abs(up);
  const R w3 = al3 * m_abs(ut), w4 = al4 * m_abs(ut);
  const R d0 = (w1 + w2) + w5;
  const R d1 = m_fma(w5, up, m_fma(w2, ut, w1 * um));
  const R d2 = m_fma(d0, vt, w3);
  const R d3 = m_fma(d0, wt, w4);
  const R d4 = m_fma(w5, H5, m_fma(w4, wt, m_fma(w3, vt, m_fma(w2, hq, w1 * H1))));
  F[0] = hs * ((L.m + Rr.m) - d0);
  F[1] = hs * ((L.F1 + Rr.F1) - d1);
  F[2] = hs * m_fma(L.m, WL[2], m_fma(Rr.m, WR[2], -d2));
  F[3] = hs * m_fma(L.m, WL[3], m_fma(Rr.m, WR[3], -d3));
  F[4] = hs * m_fma(L.m, L.H, m_fma(Rr.m, Rr.H, -d4));
  return ok;
}
// out-of-line flux of solver `mode` (1 HLLE, 2 HLLC, 3 exact) for the rare paths
template <class R> __device__ __forceinline__ void lean_fallback_call(const V5<R>& WL, const V5<R>& WR, const Par<R>& p, int mode, Cnt& c, V5<R>& F);
// Roe failed at this face: count it and replace the flux by the fallback solver's
template <class R> __device__ __forceinline__ void lean_roe_failed(const V5<R>& WL, const V5<R>& WR, const Par<R>& p, Cnt& c, V5<R>& F) {
  c.roe_fb++;
  lean_fallback_call(WL, WR, p, p.roe_fallback, c, F);
}
template <class R> __device__ __forceinline__ void lean_fallback_call(const V5<R>& WL, const V5<R>& WR, const Par<R>& p, int mode, Cnt& c, V5<R>& F) {
  FluxRet<R> r;
  if (sizeof(R) == 4) {
    r = roe_fallback_flux<R>(WL[0], WL[1], WL[2], WL[3], WL[4], WR[0], WR[1], WR[2], WR[3], WR[4], p.gamma, p.gm1, p.igm1, mode);
  } else {
    V5<R> l = WL, rr = WR;  // copies: only this branch puts its arguments on the stack
    r = roe_fallback_flux_p<R>(&l, &rr, p.gamma, p.gm1, p.igm1, mode);
  }
  F[0] = r.f0; F[1] = r.f1; F[2] = r.f2; F[3] = r.f3; F[4] = r.f4;
  c.exact += r.ex;
}
template <class R> __device__ __forceinline__ V5<R> lean_roe(const V5<R>& WL, const V5<R>& WR, const Par<R>& p, Cnt& c) {
  V5<R> F;
  if (!lean_roe_core(WL, WR, p, F)) lean_roe_failed(WL, WR, p, c, F);
  return F;
}
// the Roe flux times `scale` (scale folded into the solver's final multiplies)
template <class R> __device__ __forceinline__ V5<R> lean_roe_scaled(const V5<R>& WL, const V5<R>& WR, const Par<R>& p, Cnt& c, R scale) {
  V5<R> F;
  if (!lean_roe_core(WL, WR, p, F, R(0.5) * scale)) {
    lean_roe_failed(WL, WR, p, c, F);
#pragma unroll
    for (int q = 0; q < 5; ++q) F[q] = scale * F[q];
  }
  return F;
}

// ---- c4: HLLE (Einfeldt 1991; S9: Roe-average and local signal speeds), normal frame
template <class R> __device__ __forceinline__ V5<R> lean_hlle(const V5<R>& WL, const V5<R>& WR, const Par<R>& p) {
  const R g1 = p.gamma * p.igm1;
  const LeanState<R> L = lean_state(WL, g1), Rr = lean_state(WR, g1);
  const R wR = Rr.sq * l_rcp(L.sq + Rr.sq);
  const R ut = m_fma(wR, WR[1] - WL[1], WL[1]), vt = m_fma(wR, WR[2] - WL[2], WL[2]), wt = m_fma(wR, WR[3] - WL[3], WL[3]);
  const R Ht = m_fma(wR, Rr.H - L.H, L.H);
  const R a = l_sqrt(p.gm1 * m_fma(R(-0.5), m_fma(wt, wt, m_fma(vt, vt, ut * ut)), Ht));
  const R cL = l_sqrt(p.gamma * WL[4] * L.ir), cR = l_sqrt(p.gamma * WR[4] * Rr.ir);
  const R bm = m_min(m_min(ut - a, WL[1] - cL), R(0)), bp = m_max(m_max(ut + a, WR[1] + cR), R(0));
  const R iw = l_rcp(bp - bm), bb = bp * bm;
  // U = (rho, m, rho v, rho w, rho H - P),  F = (m, m u + P, m v, m w, m H)
  V5<R> F;
  F[0] = (m_fma(bp, L.m, -bm * Rr.m) + bb * (WR[0] - WL[0])) * iw;
  F[1] = (m_fma(bp, L.F1, -bm * Rr.F1) + bb * (Rr.m - L.m)) * iw;
  F[2] = (m_fma(bp, L.m * WL[2], -bm * (Rr.m * WR[2])) + bb * m_fma(WR[0], WR[2], -WL[0] * WL[2])) * iw;
  F[3] = (m_fma(bp, L.m * WL[3], -bm * (Rr.m * WR[3])) + bb * m_fma(WR[0], WR[3], -WL[0] * WL[3])) * iw;
  const R EL = m_fma(WL[0], L.H, -WL[4]), ER = m_fma(WR[0], Rr.H, -WR[4]);
  F[4] = (m_fma(bp, L.m * L.H, -bm * (Rr.m * Rr.H)) + bb * (ER - EL)) * iw;
  return F;
}

// ---- c4: exact solver (Toro ch. 4; S11): the same pressure function, Newton iteration, tolerance, iteration cap and
// sampling as hydro_math.cuh `exact`, organised for the GPU ("much more time-consuming"; it is config 5):
//   * fully inlined, everything in registers (the round-1 version was an out-of-line call with pointer arguments);
//   * powers as (p/P_K)^e = ex2(e lg2(p / P_K)), evaluated only on a side that is a rarefaction (with about one evaluation per
//     solve, hoisting lg2 P_K out of the iteration cost more than it saved: in fp64 log2 was 19 % of the kernel's instructions).
//     fp32 uses the SFU lg2 / ex2 approximations (relative error of z ~ 3e-8, far inside the 1e-6 tolerance);
//   * the shock branch needs one rsqrt per evaluation: sqrt(A_K / (p + B_K)) = sqrt(A_K) rsqrt(p + B_K);
//   * Halley's third-order iteration (f'' costs four more multiplies per side) and no evaluation at the accepted iterate: a step
//     delta below 4e-3 p (fp32) / 2e-5 p (fp64) is accepted with f(p + delta) = f + f' delta + f'' delta^2 / 2 and z likewise, errors
//     of order (delta/p)^3 -- so that smooth data need ONE evaluation per solve (plus one fp32 evaluation for the fp64 start).
template <class R> __device__ __forceinline__ R l_lg2(R x);
template <class R> __device__ __forceinline__ R l_ex2(R x);
#if HYDRO_F32_IEEE
template <> __device__ __forceinline__ float l_lg2<float>(float x) { return log2f(x); }
template <> __device__ __forceinline__ float l_ex2<float>(float x) { return exp2f(x); }
#else
template <> __device__ __forceinline__ float l_lg2<float>(float x) { float r; asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
template <> __device__ __forceinline__ float l_ex2<float>(float x) { float r; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
#endif
template <> __device__ __forceinline__ double l_lg2<double>(double x) { return log2(x); }
template <> __device__ __forceinline__ double l_ex2<double>(double x) { return exp2(x); }

// r^e for the exact solver's rarefaction branch.  fp32: the SFU pair.  fp64: log2 / exp2 are ~80 instructions (22 % of the config-5
// kernel's); where r is within 1/8 of one -- smooth flow, i.e. nearly every face -- the power comes from two short series instead:
// ln r = 2 atanh(s), s = (r - 1) / (r + 1), |s| <= 1/15: seven terms (remainder < 1e-18); exp(x), |x| = e |ln r| < 0.06: ten terms
// (remainder < 1e-20).  24 FP64-pipe instructions, relative error ~1e-16.
__device__ __forceinline__ float l_powr(float r, float e) { return l_ex2<float>(e * l_lg2<float>(r)); }
__device__ __forceinline__ double l_powr(double r, double e) {
  const double y = r - 1.0;
  if (fabs(y) < 0.125) {
    const double sx = y * l_rcp(r + 1.0), s2 = sx * sx;
    double a = fma(s2, 1.0 / 13.0, 1.0 / 11.0);
    a = fma(a, s2, 1.0 / 9.0);
    a = fma(a, s2, 1.0 / 7.0);
    a = fma(a, s2, 1.0 / 5.0);
    a = fma(a, s2, 1.0 / 3.0);
    a = fma(a * s2, sx, sx);                 // atanh(s)
    const double x = (e + e) * a;            // e ln r
    double b = fma(x, 1.0 / 3628800.0, 1.0 / 362880.0);
    b = fma(b, x, 1.0 / 40320.0);
    b = fma(b, x, 1.0 / 5040.0);
    b = fma(b, x, 1.0 / 720.0);
    b = fma(b, x, 1.0 / 120.0);
    b = fma(b, x, 1.0 / 24.0);
    b = fma(b, x, 1.0 / 6.0);
    b = fma(b, x, 0.5);
    b = fma(b, x, 1.0);
    return fma(b, x, 1.0);
  }
  return exp2(e * log2(r));
}

template <class R> struct ExactSide { R rho, u, P, c, irc, sA, B, k, iP; };
template <class R> struct ExactConst { R gamma, gm1, igm1, ig1, mu, e1, sA0; };  // ig1 = 1/(g+1), mu = (g-1)/(g+1), e1 = (g-1)/(2g), sA0 = sqrt(2/(g+1))
template <class R> __device__ __forceinline__ ExactConst<R> exact_const(R gamma, R gm1, R igm1, R ig1, R ig2, R sA0) {
  ExactConst<R> k;
  k.gamma = gamma; k.gm1 = gm1; k.igm1 = igm1;
  k.ig1 = ig1;
  k.mu = gm1 * ig1;
  k.e1 = gm1 * ig2;
  k.sA0 = sA0;
  return k;
}
template <class R> __device__ __forceinline__ ExactSide<R> exact_side(R rho, R u, R P, const ExactConst<R>& k) {
  ExactSide<R> s;
  s.rho = rho; s.u = u; s.P = P;
  const R gP = k.gamma * P;
  s.irc = l_rsqrt(gP * rho);                      // 1 / (rho c)
  s.c = gP * s.irc;
  s.sA = k.sA0 * l_rsqrt(rho);                    // sqrt(A_K), A_K = 2 / ((g+1) rho)
  s.B = k.mu * P;                                 // (g-1)/(g+1) P
  s.k = (s.c + s.c) * k.igm1;                     // 2 c / (g-1)
  s.iP = l_rcp(P);
  return s;
}
// f_K(p), f_K'(p), f_K''(p) and, on the rarefaction branch, z = (p/P_K)^e1 (else 0); ips = 1/p.  f_K is C^2 across
// p = P_K (both branches give f'' = -(g+1) / (2 g P_K rho_K c_K) there).
template <class R> __device__ __forceinline__ void exact_fn(R ps, R ips, const ExactSide<R>& s, R e1, R& f, R& df, R& ddf, R& z) {
  if (LEAN_EXACT_SELECT && sizeof(R) == 4) {
  // fp32: both branches on every lane, then selects: a warp meets both branches at nearly every evaluation anyway, and without
  // the branch the four chains of an evaluation (two sides x two branches) interleave (2.89 -> 2.85 ms; fp64 measured no gain)
  const R rs = l_rsqrt(ps + s.B), q = s.sA * rs, d = ps - s.P, iu = rs * rs, di = d * iu;
  const R zr = l_powr(ps * s.iP, e1);
  const R dfr = (zr * s.P * ips) * s.irc;
  const bool shock = ps > s.P;
  f = shock ? d * q : s.k * (zr - R(1));
  df = shock ? q * m_fma(R(-0.5), di, R(1)) : dfr;
  ddf = shock ? -(q * iu) * m_fma(R(-0.75), di, R(1)) : (e1 - R(1)) * (dfr * ips);
  z = shock ? R(0) : zr;
  return;
  }
  if (ps > s.P) {
    const R rs = l_rsqrt(ps + s.B), q = s.sA * rs, d = ps - s.P, iu = rs * rs, di = d * iu;
    f = d * q;
    df = q * m_fma(R(-0.5), di, R(1));
    ddf = -(q * iu) * m_fma(R(-0.75), di, R(1));
    z = R(0);
  } else {
    z = l_powr(ps * s.iP, e1);  // the power of the RATIO, taken only where a rarefaction needs it
    f = s.k * (z - R(1));
    df = (z * s.P * ips) * s.irc;
    ddf = (e1 - R(1)) * (df * ips);
  }
}
// Iteration on F(p) = f_L + f_R + du = 0 from ps (S11: negative iterate -> eps_p, at most 40 evaluations; S28: Halley's
// third-order step delta = -t / (1 - t F'' / (2 F')), t = F / F', instead of Newton's -t -- F is increasing and concave, the root
// unique).  An iterate is ACCEPTED without evaluating F there once the step is small enough for the cubic remainder to be
// negligible: |delta| < stop * p, error of p + delta of order (delta/p)^3 p.  Returns the last evaluated point ps with f, f',
// f'', z of both sides there and the step delta to the accepted iterate.
template <class R> struct ExactIter { R ps, dlt, ips, fL, dL, eL, zL, fR, dR, eR, zR; bool conv; };
template <class R> __device__ __forceinline__ ExactIter<R> exact_newton(const ExactSide<R>& L, const ExactSide<R>& Rs, R du, R e1, R epsp, R ps, R stop) {
  ExactIter<R> r;
  r.conv = false;
  r.dlt = R(0);
#pragma unroll 1
  for (int it = 0; it < 40; ++it) {
    r.ips = l_rcp(ps);
    exact_fn(ps, r.ips, L, e1, r.fL, r.dL, r.eL, r.zL);
    exact_fn(ps, r.ips, Rs, e1, r.fR, r.dR, r.eR, r.zR);
    const R idF = l_rcp(r.dL + r.dR), t = ((r.fL + r.fR) + du) * idF;
    R den = m_fma(R(-0.5) * t, (r.eL + r.eR) * idF, R(1));
    if (!(den > R(0.5))) den = R(1);                 // far from the root: a plain Newton step
    R pn = ps - l_div(t, den);
    if (!(pn > R(0))) pn = epsp;
    r.dlt = pn - ps;
    if (m_abs(r.dlt) < stop * ps) { r.conv = true; break; }
    ps = pn;
  }
  r.ps = ps;
  if (!r.conv) r.dlt = R(0);  // 40 evaluations without convergence: the last evaluated iterate stands
  return r;
}
// Acceptance rule (S28).  The accepted iterate ps + delta misses the root by about (delta/p)^3 p (Halley is cubic; the constant is
// of order one for this F).  fp32: |delta| < 4e-3 p puts it within 1e-7 p, inside the oracle's tolerance 1e-6 (S11).  fp64: S11's
// 1e-12 bounds the error of p*; |delta| < 2e-5 p gives 1e-14 p.  The fp64 iteration starts from the root of the fp32 iteration on
// the rounded states (~1e-6 p away), so that ONE fp64 evaluation suffices.
template <class R> struct ExactStop;
template <> struct ExactStop<float> { static __device__ __forceinline__ float v() { return 4e-3f; } };
template <> struct ExactStop<double> { static __device__ __forceinline__ double v() { return 2e-5; } };

template <class R> __device__ __forceinline__ V5<R> lean_exact(const V5<R>& WL, const V5<R>& WR, const Par<R>& p, Cnt& c) {
  const R g = p.gamma;
  const ExactConst<R> k = exact_const<R>(g, p.gm1, p.igm1, p.ig1, p.ig2, p.sA0);
  const R ig1 = k.ig1, mu = k.mu, e1 = k.e1;
  const ExactSide<R> L = exact_side(WL[0], WL[1], WL[4], k), Rs = exact_side(WR[0], WR[1], WR[4], k);
  const R du = Rs.u - L.u;
  V5<R> F;
  if ((L.k + Rs.k) <= du) {  // vacuum generation -> HLLE flux (S11); rare, out of line
    c.exact++;
    lean_fallback_call(WL, WR, p, 1, c, F);
    return F;
  }
  const R epsp = R(1e-6) * m_min(L.P, Rs.P);
  const R ppv = R(0.5) * (L.P + Rs.P) - R(0.125) * du * (L.rho + Rs.rho) * (L.c + Rs.c);
  R ps = m_max(epsp, ppv);
  if (sizeof(R) == 8) {  // fp64: start from the fp32 root (any start is allowed: the root is unique, f is monotone and concave)
    const ExactConst<float> kf = exact_const<float>((float)g, (float)p.gm1, (float)p.igm1, (float)p.ig1, (float)p.ig2, (float)p.sA0);
    const ExactSide<float> Lf = exact_side((float)WL[0], (float)WL[1], (float)WL[4], kf),
                           Rf = exact_side((float)WR[0], (float)WR[1], (float)WR[4], kf);
    const ExactIter<float> rf = exact_newton<float>(Lf, Rf, (float)du, kf.e1, (float)epsp, (float)ps, ExactStop<float>::v());
    const R pf = (R)(rf.ps + rf.dlt);
    if (pf > epsp && pf < R(3.0e38)) ps = pf;  // finite and positive in fp32's range; otherwise keep the linearised guess
  }
  const ExactIter<R> it = exact_newton<R>(L, Rs, du, e1, epsp, ps, ExactStop<R>::v());
  if (!it.conv) c.exact++;
  ps = it.ps;
  R fL = it.fL, fR = it.fR;
  const R dL = it.dL, dR = it.dR, zL = it.zL, zR = it.zR, dlt = it.dlt, ips = it.ips;
  // second-order update of the last evaluation to the accepted iterate ps + dlt (error of order (dlt/p)^3, as the iterate's own)
  const R hd = R(0.5) * dlt;
  fL = m_fma(m_fma(it.eL, hd, dL), dlt, fL);
  fR = m_fma(m_fma(it.eR, hd, dR), dlt, fR);
  const R x = dlt * ips;
  const R zs = m_fma(m_fma(R(0.5) * (e1 - R(1)), x, R(1)), e1 * x, R(1));  // z(ps + dlt) / z(ps) = (1 + x)^e1 to second order
  const R pst = ps + dlt;
  const R us = R(0.5) * (L.u + Rs.u) + R(0.5) * (fR - fL);
  // sample at x/t = 0 on the side of the contact given by sign(u*) (S19: u* = 0 -> left); right side mirrored
  const bool left = us >= R(0);
  const R sg = left ? R(1) : R(-1);
  const R rK = left ? L.rho : Rs.rho, PK = left ? L.P : Rs.P, cK = left ? L.c : Rs.c, vK = left ? L.u : Rs.u;
  const R ircK = left ? L.irc : Rs.irc, zE = left ? zL : zR;
  const R pr = pst * (left ? L.iP : Rs.iP);
  // z at the accepted iterate.  If the last evaluation took the shock branch (zE = 0) while the accepted iterate is a
  // rarefaction, p* lies within one accepted step (< stop p) of P_K and z = (1 + y)^e1, y = p*/P_K - 1, to second order
  const R y = pr - R(1);
  const R zK = zE > R(0) ? zE * zs : m_fma(m_fma(R(0.5) * (e1 - R(1)), y, R(1)), e1 * y, R(1));
  V5<R> W;
  W[2] = left ? WL[2] : WR[2];
  W[3] = left ? WL[3] : WR[3];
  if (pst > PK) {  // shock
    const R ig2 = p.ig2;
    const R S = vK - sg * cK * l_sqrt(m_fma((g + R(1)) * ig2, pr, p.gm1 * ig2));
    const bool undisturbed = left ? (S >= R(0)) : (S <= R(0));
    if (undisturbed) { W[0] = rK; W[1] = vK; W[4] = PK; }
    else { W[0] = l_div(rK * (pr + mu), m_fma(mu, pr, R(1))); W[1] = us; W[4] = pst; }
  } else {  // rarefaction
    const R head = vK - sg * cK, tail = us - sg * (cK * zK);
    const bool before_head = left ? (head >= R(0)) : (head <= R(0));
    const bool behind_tail = left ? (tail <= R(0)) : (tail >= R(0));
    if (before_head) { W[0] = rK; W[1] = vK; W[4] = PK; }
    else if (behind_tail) { W[0] = l_div(rK * pr, zK * zK); W[1] = us; W[4] = pst; }
    else {
      const R phi = (ig1 + ig1) + (sg * mu * vK) * (rK * ircK);  // 1 / c_K = rho_K / (rho_K c_K)
      const R wf = l_ex2((R(2) * p.igm1) * l_lg2(phi));
      W[0] = rK * wf;
      W[1] = (ig1 + ig1) * (sg * cK + R(0.5) * p.gm1 * vK);
      W[4] = PK * (phi * phi) * wf;
    }
  }
  return phys_flux(W, p);
}

// ---- c4: HLLC, Toro's pressure-based speeds (S9), select form ----------------------------------
template <class R> __device__ __forceinline__ V5<R> lean_hllc(const V5<R>& WL, const V5<R>& WR, const Par<R>& p) {
  const R g = p.gamma;
  const R irL = l_rcp(WL[0]), irR = l_rcp(WR[0]);
  const R cL = l_sqrt(g * WL[4] * irL), cR = l_sqrt(g * WR[4] * irR);
  const R ppv = R(0.5) * (WL[4] + WR[4]) - R(0.125) * (WR[1] - WL[1]) * (WL[0] + WR[0]) * (cL + cR);
  const R ps = m_max(R(0), ppv);
  const R gf = (g + R(1)) * (R(0.5) * l_rcp(g));
  const R qL = (ps <= WL[4]) ? R(1) : l_sqrt(m_fma(gf, l_div(ps, WL[4]) - R(1), R(1)));
  const R qR = (ps <= WR[4]) ? R(1) : l_sqrt(m_fma(gf, l_div(ps, WR[4]) - R(1), R(1)));
  const R SL = m_fma(-cL, qL, WL[1]), SR = m_fma(cR, qR, WR[1]);
  const R mL = WL[0] * (SL - WL[1]), mR = WR[0] * (SR - WR[1]);
  const R Ss = l_div((WR[4] - WL[4]) + WL[1] * mL - WR[1] * mR, mL - mR);
  // F_L if S_L >= 0, F_R if S_R <= 0, else the star state on the side of the contact (S19: S* = 0 -> left)
  const bool supL = SL >= R(0), supR = SR <= R(0);
  const bool left = supL || (!supR && Ss >= R(0));
  const bool star = !supL && !supR;
  const R rK = left ? WL[0] : WR[0], uK = left ? WL[1] : WR[1], vK = left ? WL[2] : WR[2], wK = left ? WL[3] : WR[3];
  const R pK = left ? WL[4] : WR[4], SK = left ? SL : SR, mK = left ? mL : mR;
  // physical flux and conserved vector of the chosen side
  const R q2 = m_fma(wK, wK, m_fma(vK, vK, uK * uK));
  const R E = m_fma(pK, p.igm1, R(0.5) * rK * q2);
  const R mom = rK * uK;
  V5<R> U, F;
  U[0] = rK; U[1] = mom; U[2] = rK * vK; U[3] = rK * wK; U[4] = E;
  F[0] = mom; F[1] = m_fma(mom, uK, pK); F[2] = mom * vK; F[3] = mom * wK; F[4] = (E + pK) * uK;
  const R f = l_div(mK, SK - Ss);
  V5<R> Us;
  Us[0] = f;
  Us[1] = f * Ss;
  Us[2] = f * vK;
  Us[3] = f * wK;
  Us[4] = f * (l_div(E, rK) + (Ss - uK) * (Ss + l_div(pK, mK)));
#pragma unroll
  for (int q = 0; q < 5; ++q) F[q] = star ? m_fma(SK, Us[q] - U[q], F[q]) : F[q];
  return F;
}

}  // namespace hydro
