// oracle/hydro_oracle.cpp
//
// TEST INFRASTRUCTURE ONLY.  Plain, slow, single-threaded-per-group CPU oracle of the
// directionally unsplit patch-group fluid update of Schive, Zhang & Chiueh (arXiv:1103.3373).
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
// load this library.  It shares no code with paper_1103_3373_b200/csrc (the CUDA path).
//
// The paper gives the method as a five-item list (section 2) plus options
// (PAPER.md:46-50); formulas are the textbook forms of the methods it cites, in the readings
// fixed by SURVEY.md section 8(c) (c0-c6) and restated in DESIGN.md ("Readings").  Each function
// cites the passage it follows.  No blocking, fusion or reordering beyond those statements:
// every stage is a plain loop over a box-shaped region of one padded patch group.
//
// Pins (tests/test_oracle_*.py, -m "not gpu"): P1-P15 of SURVEY.md 8(c).
// parity unpinned: S5 (tracing variant), S6 (PPM variant), S7 (theta), S9 (HLL wave speeds),
// S10 (Roe fallback choice), S11 (exact-solver constants), S14 (floors) -- several choices are
// all "correct" (each passes P1-P15); they are fixed by DESIGN.md only.
//
// Build: g++ -O2 -ffp-contract=off -fopenmp -shared -fPIC (see oracle/build_oracle.py).
// OpenMP is used ONLY as a parallel-for over independent patch groups (patch-level
// parallelism); nthreads=1 is the single-threaded oracle.

#include <algorithm>
#include <array>
#include <cmath>
#include <cstddef>
#include <cstring>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

constexpr int PS = 16;  // interior cells per side of a patch group (2x2x2 patches of 8^3)

template <class R> using V5 = std::array<R, 5>;

// status counters (host side): [0] Roe fallbacks, [1] non-positive rho/P seen in con->prim,
// [2] exact-solver non-convergence / vacuum, [3] Riemann solves (all), [4] Riemann solves on faces
// owned by an interior cell (f in [0,16), transverse in [0,16)^2) -- the per-cell count of PAPER.md:35,105.
struct Status {
  long long c[8] = {0, 0, 0, 0, 0, 0, 0, 0};
};

template <class R> struct Params {
  R gamma, nu;      // nu = dt/dh
  int scheme;       // 0 MHM, 1 VL, 2 CTU
  int riemann;      // 0 exact, 1 HLLE, 2 HLLC, 3 Roe
  int limiter;      // 0 generalized minmod, 1 van Leer, 2 van Albada, 3 hybrid
  int recon;        // 0 PLM, 1 PPM
  int char_limit;   // 0 primitive, 1 characteristic variables
  int roe_fallback; // 1 HLLE, 2 HLLC, 3 exact
  R theta;          // generalized-minmod coefficient
  R min_dens, min_pres;  // 0 => no floor
};

// ---------------------------------------------------------------------------------------------
// c0. Conversions (ideal gas, "adiabatic hydrodynamic" PAPER.md:11).
// U = (rho, rho vx, rho vy, rho vz, E), W = (rho, vx, vy, vz, P), E = P/(gamma-1) + rho|v|^2/2.
template <class R> V5<R> cons2prim(const V5<R>& U, const Params<R>& p, Status* st) {
  R rho = U[0];
  if (p.min_dens > R(0) && rho < p.min_dens) rho = p.min_dens;
  const R vx = U[1] / rho, vy = U[2] / rho, vz = U[3] / rho;
  R P = (p.gamma - R(1)) * (U[4] - R(0.5) * rho * ((vx * vx + vy * vy) + vz * vz));
  if (st && (!(U[0] > R(0)) || !(P > R(0)))) st->c[1]++;
  if (p.min_pres > R(0) && P < p.min_pres) P = p.min_pres;
  return {rho, vx, vy, vz, P};
}
template <class R> V5<R> prim2cons(const V5<R>& W, R gamma) {
  const R rho = W[0];
  const R E = W[4] / (gamma - R(1)) + R(0.5) * rho * ((W[1] * W[1] + W[2] * W[2]) + W[3] * W[3]);
  return {rho, rho * W[1], rho * W[2], rho * W[3], E};
}

// Normal-frame relabelling ("(n,t1,t2) = (x,y,z), (y,z,x), (z,x,y)").
// Works for primitive, conserved and flux 5-vectors alike: slot 1+d <-> slot 1, etc.
template <class R> V5<R> to_normal(const V5<R>& a, int d) {
  return {a[0], a[1 + d], a[1 + (d + 1) % 3], a[1 + (d + 2) % 3], a[4]};
}
template <class R> V5<R> from_normal(const V5<R>& n, int d) {
  V5<R> a;
  a[0] = n[0];
  a[1 + d] = n[1];
  a[1 + (d + 1) % 3] = n[2];
  a[1 + (d + 2) % 3] = n[3];
  a[4] = n[4];
  return a;
}

// Physical flux of a normal-frame primitive state:
// F(W) = (rho vn, rho vn^2 + P, rho vn vt1, rho vn vt2, (E+P) vn).
template <class R> V5<R> phys_flux(const V5<R>& W, R gamma) {
  const R rho = W[0], vn = W[1], v1 = W[2], v2 = W[3], P = W[4];
  const R E = P / (gamma - R(1)) + R(0.5) * rho * ((vn * vn + v1 * v1) + v2 * v2);
  return {rho * vn, rho * vn * vn + P, rho * vn * v1, rho * vn * v2, (E + P) * vn};
}
template <class R> V5<R> cons_n(const V5<R>& W, R gamma) {  // normal-frame conserved vector
  const R rho = W[0];
  const R E = W[4] / (gamma - R(1)) + R(0.5) * rho * ((W[1] * W[1] + W[2] * W[2]) + W[3] * W[3]);
  return {rho, rho * W[1], rho * W[2], rho * W[3], E};
}

// ---------------------------------------------------------------------------------------------
// c1. Slope limiters (PAPER.md:48 names them; Toro-style definitions).
template <class R> R limited_slope(R dL, R dR, R dC, int limiter, R theta) {
  if (dL * dR <= R(0)) return R(0);  // tie-break S19: zero product -> zero slope
  const R s = (dC > R(0)) ? R(1) : R(-1);
  const R aL = std::fabs(dL), aR = std::fabs(dR), aC = std::fabs(dC);
  switch (limiter) {
    case 0: return s * std::min(std::min(theta * aL, theta * aR), aC);          // generalized minmod
    case 1: return R(2) * dL * dR / (dL + dR);                                 // van Leer
    case 2: return dL * dR * (dL + dR) / (dL * dL + dR * dR);                  // van Albada
    default: {                                                                 // Athena hybrid
      const R vl = std::fabs(R(2) * dL * dR / (dL + dR));
      return s * std::min(std::min(R(2) * aL, R(2) * aR), std::min(aC, vl));
    }
  }
}

// Eigen-system of the primitive normal-direction Jacobian at W.
// Waves 1..5 with speeds vn-c, vn, vn, vn, vn+c.
template <class R> V5<R> eig_project(const V5<R>& W, R c, const V5<R>& d) {  // L . d
  const R c2 = c * c;
  return {R(0.5) * (d[4] / c2 - W[0] * d[1] / c), d[0] - d[4] / c2, d[2], d[3],
          R(0.5) * (d[4] / c2 + W[0] * d[1] / c)};
}
template <class R> V5<R> eig_expand(const V5<R>& W, R c, const V5<R>& a) {  // sum_a a_a R_a
  return {(a[0] + a[1]) + a[4], (c / W[0]) * (a[4] - a[0]), a[2], a[3], (c * c) * (a[0] + a[4])};
}

// Limited slope vector of the middle cell of (Wm, W0, Wp), all normal-frame primitives.
template <class R> V5<R> slope_vec(const V5<R>& Wm, const V5<R>& W0, const V5<R>& Wp, const Params<R>& p) {
  V5<R> dL, dR, dC, out;
  for (int q = 0; q < 5; ++q) {
    dL[q] = W0[q] - Wm[q];
    dR[q] = Wp[q] - W0[q];
    dC[q] = R(0.5) * (dL[q] + dR[q]);
  }
  if (p.char_limit) {  // S8: project dL, dR, dC with the eigenvectors of W0, limit, project back
    const R c = std::sqrt(p.gamma * W0[4] / W0[0]);
    const V5<R> aL = eig_project(W0, c, dL), aR = eig_project(W0, c, dR), aC = eig_project(W0, c, dC);
    V5<R> a;
    for (int q = 0; q < 5; ++q) a[q] = limited_slope(aL[q], aR[q], aC[q], p.limiter, p.theta);
    return eig_expand(W0, c, a);
  }
  for (int q = 0; q < 5; ++q) out[q] = limited_slope(dL[q], dR[q], dC[q], p.limiter, p.theta);
  return out;
}

// ---------------------------------------------------------------------------------------------
// c2 + c3. Face values of cell i from the normal-frame pencil Wn[i-2..i+2] (PLM uses +-1 only).
// Wlo = W^- at the lower face, Wup = W^+ at the upper face.  trace => CTU characteristic
// tracing to dt/2, reference-state form with approaching waves only (S5).
template <class R>
void reconstruct(const V5<R>* Wc /* points at cell i; Wc[-2..2] valid for PPM, [-1..1] for PLM */,
                 const Params<R>& p, bool trace, V5<R>& Wlo, V5<R>& Wup) {
  const V5<R>& W0 = Wc[0];
  const R nu = p.nu;
  V5<R> dW = slope_vec(Wc[-1], Wc[0], Wc[1], p);
  V5<R> WL, WR, D, W6;
  if (p.recon == 0) {  // PLM (c2)
    for (int q = 0; q < 5; ++q) {
      WL[q] = W0[q] - R(0.5) * dW[q];
      WR[q] = W0[q] + R(0.5) * dW[q];
    }
  } else {  // PPM, Colella-Woodward interpolation + monotonisation, no steepening/flattening (S6)
    const V5<R> dWm = slope_vec(Wc[-2], Wc[-1], Wc[0], p);
    const V5<R> dWp = slope_vec(Wc[0], Wc[1], Wc[2], p);
    for (int q = 0; q < 5; ++q) {
      R wl = R(0.5) * (Wc[-1][q] + W0[q]) - (dW[q] - dWm[q]) / R(6);
      R wr = R(0.5) * (W0[q] + Wc[1][q]) - (dWp[q] - dW[q]) / R(6);
      const R w0 = W0[q];
      if ((wr - w0) * (w0 - wl) <= R(0)) {
        wl = w0;
        wr = w0;
      } else {
        const R dd = wr - wl, m = w0 - R(0.5) * (wl + wr);
        if (R(6) * dd * m > dd * dd) wl = R(3) * w0 - R(2) * wr;
        else if (R(6) * dd * m < -(dd * dd)) wr = R(3) * w0 - R(2) * wl;
      }
      WL[q] = wl;
      WR[q] = wr;
      D[q] = wr - wl;
      W6[q] = R(6) * (w0 - R(0.5) * (wl + wr));
    }
  }
  if (!trace) {
    Wlo = WL;
    Wup = WR;
    return;
  }
  // c3: characteristic tracing.
  const R c = std::sqrt(p.gamma * W0[4] / W0[0]);
  const R lam[5] = {W0[1] - c, W0[1], W0[1], W0[1], W0[1] + c};
  const R lamM = lam[4], lam0 = lam[0];
  if (p.recon == 0) {
    const V5<R> a = eig_project(W0, c, dW);
    V5<R> ap = {0, 0, 0, 0, 0}, am = {0, 0, 0, 0, 0};
    for (int k = 0; k < 5; ++k) {
      if (lam[k] > R(0)) ap[k] = R(0.5) * nu * (lamM - lam[k]) * a[k];
      if (lam[k] < R(0)) am[k] = R(0.5) * nu * (lam0 - lam[k]) * a[k];
    }
    const V5<R> sp = eig_expand(W0, c, ap), sm = eig_expand(W0, c, am);
    const R fp = R(0.5) * nu * std::max(lamM, R(0)), fm = R(0.5) * nu * std::min(lam0, R(0));
    for (int q = 0; q < 5; ++q) {
      Wup[q] = (WR[q] - fp * dW[q]) + sp[q];
      Wlo[q] = (WL[q] - fm * dW[q]) + sm[q];
    }
  } else {
    const R sgp = nu * std::max(lamM, R(0)), sgm = nu * std::min(lam0, R(0));
    V5<R> tp, tm;  // vectors whose characteristic projections are summed over approaching waves
    V5<R> DmW6, DpW6;
    for (int q = 0; q < 5; ++q) {
      DmW6[q] = D[q] - W6[q];
      DpW6[q] = D[q] + W6[q];
    }
    const V5<R> aDm = eig_project(W0, c, DmW6), aDp = eig_project(W0, c, DpW6), a6 = eig_project(W0, c, W6);
    V5<R> ap = {0, 0, 0, 0, 0}, am = {0, 0, 0, 0, 0};
    for (int k = 0; k < 5; ++k) {
      if (lam[k] > R(0)) {
        const R A = R(0.5) * nu * (lamM - lam[k]);
        const R B = (nu * nu / R(3)) * (lamM * lamM - lam[k] * lam[k]);
        ap[k] = A * aDm[k] + B * a6[k];
      }
      if (lam[k] < R(0)) {
        const R C = R(0.5) * nu * (lam0 - lam[k]);
        const R Dk = (nu * nu / R(3)) * (lam0 * lam0 - lam[k] * lam[k]);
        am[k] = C * aDp[k] + Dk * a6[k];
      }
    }
    tp = eig_expand(W0, c, ap);
    tm = eig_expand(W0, c, am);
    for (int q = 0; q < 5; ++q) {
      Wup[q] = (WR[q] - R(0.5) * sgp * (D[q] - (R(1) - R(2) / R(3) * sgp) * W6[q])) + tp[q];
      Wlo[q] = (WL[q] - R(0.5) * sgm * (D[q] + (R(1) + R(2) / R(3) * sgm) * W6[q])) + tm[q];
    }
  }
}

// ---------------------------------------------------------------------------------------------
// c4. Riemann solvers, normal frame (rho, vn, vt1, vt2, P) -> (F_rho, F_mn, F_mt1, F_mt2, F_E).
template <class R> struct RoeAvg {
  R vn, v1, v2, H, a;
};
template <class R> RoeAvg<R> roe_average(const V5<R>& WL, const V5<R>& WR, R gamma) {
  const V5<R> UL = cons_n(WL, gamma), UR = cons_n(WR, gamma);
  const R HL = (UL[4] + WL[4]) / WL[0], HR = (UR[4] + WR[4]) / WR[0];
  const R sL = std::sqrt(WL[0]), sR = std::sqrt(WR[0]), den = sL + sR;
  RoeAvg<R> r;
  r.vn = (sL * WL[1] + sR * WR[1]) / den;
  r.v1 = (sL * WL[2] + sR * WR[2]) / den;
  r.v2 = (sL * WL[3] + sR * WR[3]) / den;
  r.H = (sL * HL + sR * HR) / den;
  const R q2 = (r.vn * r.vn + r.v1 * r.v1) + r.v2 * r.v2;
  r.a = std::sqrt((gamma - R(1)) * (r.H - R(0.5) * q2));
  return r;
}

// HLLE (Einfeldt 1991).
template <class R> V5<R> hlle(const V5<R>& WL, const V5<R>& WR, const Params<R>& p) {
  const R g = p.gamma;
  const RoeAvg<R> r = roe_average(WL, WR, g);
  const R cL = std::sqrt(g * WL[4] / WL[0]), cR = std::sqrt(g * WR[4] / WR[0]);
  const R SL = std::min(r.vn - r.a, WL[1] - cL), SR = std::max(r.vn + r.a, WR[1] + cR);
  const R bm = std::min(SL, R(0)), bp = std::max(SR, R(0));
  const V5<R> UL = cons_n(WL, g), UR = cons_n(WR, g), FL = phys_flux(WL, g), FR = phys_flux(WR, g);
  V5<R> F;
  for (int q = 0; q < 5; ++q) F[q] = ((bp * FL[q] - bm * FR[q]) + bp * bm * (UR[q] - UL[q])) / (bp - bm);
  return F;
}

// HLLC with Toro's pressure-based wave speeds.
template <class R> V5<R> hllc(const V5<R>& WL, const V5<R>& WR, const Params<R>& p) {
  const R g = p.gamma;
  const R cL = std::sqrt(g * WL[4] / WL[0]), cR = std::sqrt(g * WR[4] / WR[0]);
  const R rb = R(0.5) * (WL[0] + WR[0]), cb = R(0.5) * (cL + cR);
  const R ppv = R(0.5) * (WL[4] + WR[4]) - R(0.5) * (WR[1] - WL[1]) * rb * cb;
  const R ps = std::max(R(0), ppv);
  const R qL = (ps <= WL[4]) ? R(1) : std::sqrt(R(1) + (g + R(1)) / (R(2) * g) * (ps / WL[4] - R(1)));
  const R qR = (ps <= WR[4]) ? R(1) : std::sqrt(R(1) + (g + R(1)) / (R(2) * g) * (ps / WR[4] - R(1)));
  const R SL = WL[1] - cL * qL, SR = WR[1] + cR * qR;
  const V5<R> UL = cons_n(WL, g), UR = cons_n(WR, g), FL = phys_flux(WL, g), FR = phys_flux(WR, g);
  if (SL >= R(0)) return FL;
  if (SR <= R(0)) return FR;
  const R mL = WL[0] * (SL - WL[1]), mR = WR[0] * (SR - WR[1]);
  const R Ss = ((WR[4] - WL[4]) + WL[1] * mL - WR[1] * mR) / (mL - mR);
  V5<R> F;
  if (Ss >= R(0)) {  // S_L < 0 <= S*  (tie S* = 0 -> left star, S19)
    const R f = mL / (SL - Ss);
    const V5<R> Us = {f, f * Ss, f * WL[2], f * WL[3],
                      f * (UL[4] / WL[0] + (Ss - WL[1]) * (Ss + WL[4] / mL))};
    for (int q = 0; q < 5; ++q) F[q] = FL[q] + SL * (Us[q] - UL[q]);
  } else {
    const R f = mR / (SR - Ss);
    const V5<R> Us = {f, f * Ss, f * WR[2], f * WR[3],
                      f * (UR[4] / WR[0] + (Ss - WR[1]) * (Ss + WR[4] / mR))};
    for (int q = 0; q < 5; ++q) F[q] = FR[q] + SR * (Us[q] - UR[q]);
  }
  return F;
}

// Exact solver (Toro ch. 4).
template <class R> struct ExactTol;
template <> struct ExactTol<double> { static constexpr double v = 1e-12; };
template <> struct ExactTol<float> { static constexpr float v = 1e-6f; };

template <class R> void pressure_fn(R p, R rhoK, R PK, R cK, R g, R& f, R& df) {
  if (p > PK) {  // shock
    const R A = R(2) / ((g + R(1)) * rhoK), B = (g - R(1)) / (g + R(1)) * PK;
    const R s = std::sqrt(A / (p + B));
    f = (p - PK) * s;
    df = s * (R(1) - (p - PK) / (R(2) * (B + p)));
  } else {  // rarefaction
    f = R(2) * cK / (g - R(1)) * (std::pow(p / PK, (g - R(1)) / (R(2) * g)) - R(1));
    df = std::pow(p / PK, -(g + R(1)) / (R(2) * g)) / (rhoK * cK);
  }
}
// star state: returns false on vacuum generation
template <class R> bool exact_star(const V5<R>& WL, const V5<R>& WR, R g, R& ps, R& us, bool& converged) {
  const R cL = std::sqrt(g * WL[4] / WL[0]), cR = std::sqrt(g * WR[4] / WR[0]);
  const R du = WR[1] - WL[1];
  converged = true;
  if (R(2) * (cL + cR) / (g - R(1)) <= du) return false;  // vacuum
  const R epsp = R(1e-6) * std::min(WL[4], WR[4]);
  const R ppv = R(0.5) * (WL[4] + WR[4]) - R(0.125) * du * (WL[0] + WR[0]) * (cL + cR);
  R p = std::max(epsp, ppv);
  R fL, dL, fR, dR;
  converged = false;
  for (int it = 0; it < 40; ++it) {
    pressure_fn(p, WL[0], WL[4], cL, g, fL, dL);
    pressure_fn(p, WR[0], WR[4], cR, g, fR, dR);
    R pn = p - ((fL + fR) + du) / (dL + dR);
    if (!(pn > R(0))) pn = epsp;
    const R chg = R(2) * std::fabs(pn - p) / (pn + p);
    p = pn;
    if (chg < ExactTol<R>::v) {
      converged = true;
      break;
    }
  }
  pressure_fn(p, WL[0], WL[4], cL, g, fL, dL);
  pressure_fn(p, WR[0], WR[4], cR, g, fR, dR);
  ps = p;
  us = R(0.5) * (WL[1] + WR[1]) + R(0.5) * (fR - fL);
  return true;
}
// sample the self-similar solution at x/t = 0.
template <class R> V5<R> exact_sample0(const V5<R>& WL, const V5<R>& WR, R g, R ps, R us) {
  const R mu = (g - R(1)) / (g + R(1));
  V5<R> W;
  if (us >= R(0)) {  // left of contact (tie u* = 0 -> left, S19)
    const R rK = WL[0], vK = WL[1], PK = WL[4], cK = std::sqrt(g * PK / rK);
    W[2] = WL[2];
    W[3] = WL[3];
    if (ps > PK) {  // left shock
      const R S = vK - cK * std::sqrt((g + R(1)) / (R(2) * g) * ps / PK + (g - R(1)) / (R(2) * g));
      if (S >= R(0)) { W[0] = rK; W[1] = vK; W[4] = PK; }
      else { W[0] = rK * (ps / PK + mu) / (mu * ps / PK + R(1)); W[1] = us; W[4] = ps; }
    } else {  // left rarefaction
      const R head = vK - cK;
      const R cs = cK * std::pow(ps / PK, (g - R(1)) / (R(2) * g));
      const R tail = us - cs;
      if (head >= R(0)) { W[0] = rK; W[1] = vK; W[4] = PK; }
      else if (tail <= R(0)) { W[0] = rK * std::pow(ps / PK, R(1) / g); W[1] = us; W[4] = ps; }
      else {
        const R phi = R(2) / (g + R(1)) + mu * vK / cK;
        W[0] = rK * std::pow(phi, R(2) / (g - R(1)));
        W[1] = R(2) / (g + R(1)) * (cK + R(0.5) * (g - R(1)) * vK);
        W[4] = PK * std::pow(phi, R(2) * g / (g - R(1)));
      }
    }
  } else {
    const R rK = WR[0], vK = WR[1], PK = WR[4], cK = std::sqrt(g * PK / rK);
    W[2] = WR[2];
    W[3] = WR[3];
    if (ps > PK) {  // right shock
      const R S = vK + cK * std::sqrt((g + R(1)) / (R(2) * g) * ps / PK + (g - R(1)) / (R(2) * g));
      if (S <= R(0)) { W[0] = rK; W[1] = vK; W[4] = PK; }
      else { W[0] = rK * (ps / PK + mu) / (mu * ps / PK + R(1)); W[1] = us; W[4] = ps; }
    } else {
      const R head = vK + cK;
      const R cs = cK * std::pow(ps / PK, (g - R(1)) / (R(2) * g));
      const R tail = us + cs;
      if (head <= R(0)) { W[0] = rK; W[1] = vK; W[4] = PK; }
      else if (tail >= R(0)) { W[0] = rK * std::pow(ps / PK, R(1) / g); W[1] = us; W[4] = ps; }
      else {
        const R phi = R(2) / (g + R(1)) - mu * vK / cK;
        W[0] = rK * std::pow(phi, R(2) / (g - R(1)));
        W[1] = R(2) / (g + R(1)) * (-cK + R(0.5) * (g - R(1)) * vK);
        W[4] = PK * std::pow(phi, R(2) * g / (g - R(1)));
      }
    }
  }
  return W;
}
template <class R> V5<R> exact(const V5<R>& WL, const V5<R>& WR, const Params<R>& p, Status* st) {
  R ps, us;
  bool conv;
  if (!exact_star(WL, WR, p.gamma, ps, us, conv)) {  // vacuum -> HLLE flux, status[2]++
    if (st) st->c[2]++;
    return hlle(WL, WR, p);
  }
  if (!conv && st) st->c[2]++;
  return phys_flux(exact_sample0(WL, WR, p.gamma, ps, us), p.gamma);
}

// Roe's solver (Roe 1981): no entropy fix; failure test on the two
// intermediate states U_L + a1 K1 and U_R - a5 K5; on failure the face flux is recomputed with
// the fallback solver ("same strategy adopted in Athena").
template <class R> V5<R> roe(const V5<R>& WL, const V5<R>& WR, const Params<R>& p, Status* st) {
  const R g = p.gamma, g1 = g - R(1);
  const RoeAvg<R> r = roe_average(WL, WR, g);
  const V5<R> UL = cons_n(WL, g), UR = cons_n(WR, g), FL = phys_flux(WL, g), FR = phys_flux(WR, g);
  const R vn = r.vn, v1 = r.v1, v2 = r.v2, H = r.H, a = r.a;
  const R q2 = (vn * vn + v1 * v1) + v2 * v2;
  V5<R> du;
  for (int q = 0; q < 5; ++q) du[q] = UR[q] - UL[q];
  const R a3 = du[2] - v1 * du[0], a4 = du[3] - v2 * du[0];
  const R du5 = (du[4] - a3 * v1) - a4 * v2;
  const R a2 = g1 / (a * a) * ((du[0] * (H - vn * vn) + vn * du[1]) - du5);
  const R a1 = ((du[0] * (vn + a) - du[1]) - a * a2) / (R(2) * a);
  const R a5 = du[0] - (a1 + a2);
  const V5<R> K1 = {R(1), vn - a, v1, v2, H - vn * a}, K2 = {R(1), vn, v1, v2, R(0.5) * q2},
              K3 = {R(0), R(0), R(1), R(0), v1}, K4 = {R(0), R(0), R(0), R(1), v2},
              K5 = {R(1), vn + a, v1, v2, H + vn * a};
  // failure detection
  bool fail = false;
  {
    V5<R> A, B;
    for (int q = 0; q < 5; ++q) {
      A[q] = UL[q] + a1 * K1[q];
      B[q] = UR[q] - a5 * K5[q];
    }
    const R PA = g1 * (A[4] - R(0.5) * ((A[1] * A[1] + A[2] * A[2]) + A[3] * A[3]) / A[0]);
    const R PB = g1 * (B[4] - R(0.5) * ((B[1] * B[1] + B[2] * B[2]) + B[3] * B[3]) / B[0]);
    if (!(A[0] > R(0)) || !(PA > R(0)) || !(B[0] > R(0)) || !(PB > R(0))) fail = true;
  }
  if (fail) {
    if (st) st->c[0]++;
    if (p.roe_fallback == 2) return hllc(WL, WR, p);
    if (p.roe_fallback == 3) return exact(WL, WR, p, st);
    return hlle(WL, WR, p);
  }
  const R l1 = std::fabs(vn - a), l2 = std::fabs(vn), l5 = std::fabs(vn + a);
  V5<R> F;
  for (int q = 0; q < 5; ++q) {
    const R diss = (((a1 * l1 * K1[q] + a2 * l2 * K2[q]) + a3 * l2 * K3[q]) + a4 * l2 * K4[q]) + a5 * l5 * K5[q];
    F[q] = R(0.5) * (FL[q] + FR[q]) - R(0.5) * diss;
  }
  return F;
}

template <class R>
V5<R> riemann(const V5<R>& WL, const V5<R>& WR, const Params<R>& p, Status* st, bool owned) {
  if (st) {
    st->c[3]++;
    if (owned) st->c[4]++;
  }
  switch (p.riemann) {
    case 0: return exact(WL, WR, p, st);
    case 1: return hlle(WL, WR, p);
    case 2: return hllc(WL, WR, p);
    default: return roe(WL, WR, p, st);
  }
}

// ---------------------------------------------------------------------------------------------
// c5. Integrators on ONE padded patch group (box of S^3 cells, S = 16 + 2g, x fastest;
// PAPER.md:58, 65, 79).  Regions are boxes in interior coordinates.
template <class R> struct Group {
  int g, S;
  size_t n;                                     // S^3
  std::vector<V5<R>> U, W;                      // conserved input, primitive
  std::vector<V5<R>> lo[3], up[3];              // face states per direction (xyz-frame primitives)
  std::vector<V5<R>> F1[3], F2[3];              // pass-1 / pass-2 fluxes; entry of cell c = its LOWER face
  std::vector<V5<R>> Uh;                        // VL half-step conserved
  explicit Group(int g_) : g(g_), S(PS + 2 * g_), n((size_t)S * S * S) {}
  inline size_t id(int i, int j, int k) const { return ((size_t)(k + g) * S + (j + g)) * S + (i + g); }
  inline size_t id(const int c[3]) const { return id(c[0], c[1], c[2]); }
};

inline bool in_interior(const int c[3], int d) {  // face owned by an interior cell
  (void)d;
  return c[0] >= 0 && c[0] < PS && c[1] >= 0 && c[1] < PS && c[2] >= 0 && c[2] < PS;
}

// face states of all cells in box [lo_, hi_]^3 (per-direction bounds) from the primitive array Wsrc
template <class R>
void recon_direction(Group<R>& G, const std::vector<V5<R>>& Wsrc, int d, const int lo_[3], const int hi_[3],
                     const Params<R>& p, bool trace) {
  V5<R> pencil[5];
  int c[3];
  for (c[2] = lo_[2]; c[2] <= hi_[2]; ++c[2])
    for (c[1] = lo_[1]; c[1] <= hi_[1]; ++c[1])
      for (c[0] = lo_[0]; c[0] <= hi_[0]; ++c[0]) {
        const int w = (p.recon == 0) ? 1 : 2;
        for (int s = -w; s <= w; ++s) {
          int cc[3] = {c[0], c[1], c[2]};
          cc[d] += s;
          pencil[2 + s] = to_normal(Wsrc[G.id(cc)], d);
        }
        V5<R> l, u;
        reconstruct(&pencil[2], p, trace, l, u);
        G.lo[d][G.id(c)] = from_normal(l, d);
        G.up[d][G.id(c)] = from_normal(u, d);
      }
}

// Riemann fluxes at the lower faces of cells in the box, from (up[d] of c - e_d, lo[d] of c)
template <class R>
void flux_direction(Group<R>& G, const std::vector<V5<R>>& up, const std::vector<V5<R>>& lo,
                    std::vector<V5<R>>& F, int d, const int lo_[3], const int hi_[3], const Params<R>& p,
                    Status* st) {
  int c[3];
  for (c[2] = lo_[2]; c[2] <= hi_[2]; ++c[2])
    for (c[1] = lo_[1]; c[1] <= hi_[1]; ++c[1])
      for (c[0] = lo_[0]; c[0] <= hi_[0]; ++c[0]) {
        int m[3] = {c[0], c[1], c[2]};
        m[d] -= 1;
        const V5<R> f = riemann(to_normal(up[G.id(m)], d), to_normal(lo[G.id(c)], d), p, st, in_interior(c, d));
        F[G.id(c)] = from_normal(f, d);
      }
}

template <class R>
void solve_group(const R* in, R* out, R* face_flux, int g, const Params<R>& p, Status* st) {
  Group<R> G(g);
  const size_t n = G.n;
  const R nu = p.nu;
  const int gmin = (p.scheme == 1 ? 3 : 2) + (p.recon == 1 ? 1 : 0);
  G.U.resize(n);
  G.W.resize(n);
  for (int d = 0; d < 3; ++d) {
    G.lo[d].resize(n);
    G.up[d].resize(n);
    G.F1[d].resize(n);
    G.F2[d].resize(n);
  }
  // (1) primitive variables on the g_min box (c0); cells outside it are never read.
  for (int k = -gmin; k < PS + gmin; ++k)
    for (int j = -gmin; j < PS + gmin; ++j)
      for (int i = -gmin; i < PS + gmin; ++i) {
        const size_t x = G.id(i, j, k);
        for (int v = 0; v < 5; ++v) G.U[x][v] = in[(size_t)v * n + x];
        G.W[x] = cons2prim(G.U[x], p, st);
      }
  const int e[3][3] = {{1, 0, 0}, {0, 1, 0}, {0, 0, 1}};
  // region of half-step / corrected face states for direction d: c_d in [-1,16], transverse in [0,16)
  auto fs_lo = [&](int d, int lo_[3], int hi_[3]) {
    for (int a = 0; a < 3; ++a) {
      lo_[a] = (a == d) ? -1 : 0;
      hi_[a] = (a == d) ? PS : PS - 1;
    }
  };
  // region of final fluxes for direction d: f_d in [0,16], transverse in [0,16)
  auto ff = [&](int d, int lo_[3], int hi_[3]) {
    for (int a = 0; a < 3; ++a) {
      lo_[a] = 0;
      hi_[a] = (a == d) ? PS : PS - 1;
    }
  };
  const int b_lo[3] = {-1, -1, -1}, b_hi[3] = {PS, PS, PS};  // [-1,16]^3

  if (p.scheme == 2) {
    // ---- CTU (Colella 1990; six-solve 3-D variant of Gardiner & Stone 2008) ----
    // (2) traced face states W^+-_d on [-1,16]^3              PAPER.md:39 step (1)
    for (int d = 0; d < 3; ++d) recon_direction(G, G.W, d, b_lo, b_hi, p, true);
    // (3) F*_d at faces f_d in [0,16], transverse in [-1,16]  PAPER.md:40 step (2)
    for (int d = 0; d < 3; ++d) {
      int lo_[3] = {-1, -1, -1}, hi_[3] = {PS, PS, PS};
      lo_[d] = 0;
      flux_direction(G, G.up[d], G.lo[d], G.F1[d], d, lo_, hi_, p, st);
    }
    // (4) transverse correction with half nu (S4)            PAPER.md:41 step (3)
    for (int d = 0; d < 3; ++d) {
      const int t1 = (d + 1) % 3, t2 = (d + 2) % 3;
      int lo_[3], hi_[3], c[3];
      fs_lo(d, lo_, hi_);
      for (c[2] = lo_[2]; c[2] <= hi_[2]; ++c[2])
        for (c[1] = lo_[1]; c[1] <= hi_[1]; ++c[1])
          for (c[0] = lo_[0]; c[0] <= hi_[0]; ++c[0]) {
            const size_t x = G.id(c);
            const int u1[3] = {c[0] + e[t1][0], c[1] + e[t1][1], c[2] + e[t1][2]};
            const int u2[3] = {c[0] + e[t2][0], c[1] + e[t2][1], c[2] + e[t2][2]};
            const V5<R>&A1 = G.F1[t1][G.id(u1)], &A0 = G.F1[t1][x], &B1 = G.F1[t2][G.id(u2)], &B0 = G.F1[t2][x];
            for (int side = 0; side < 2; ++side) {
              std::vector<V5<R>>& fs = side ? G.up[d] : G.lo[d];
              V5<R> Uc = prim2cons(fs[x], p.gamma);
              for (int q = 0; q < 5; ++q) Uc[q] = Uc[q] - R(0.5) * nu * ((A1[q] - A0[q]) + (B1[q] - B0[q]));
              fs[x] = cons2prim(Uc, p, st);
            }
          }
    }
  } else if (p.scheme == 0) {
    // ---- MHM (MUSCL-Hancock; S13) ----
    // (2) untraced face states on [-1,16]^3, all directions
    for (int d = 0; d < 3; ++d) recon_direction(G, G.W, d, b_lo, b_hi, p, false);
    // (3) one cell-local increment from the physical fluxes of the cell's own six face values
    std::vector<V5<R>> inc(n);
    {
      int c[3];
      for (c[2] = -1; c[2] <= PS; ++c[2])
        for (c[1] = -1; c[1] <= PS; ++c[1])
          for (c[0] = -1; c[0] <= PS; ++c[0]) {
            const size_t x = G.id(c);
            V5<R> dF[3];
            for (int d = 0; d < 3; ++d) {
              const V5<R> fu = from_normal(phys_flux(to_normal(G.up[d][x], d), p.gamma), d);
              const V5<R> fl = from_normal(phys_flux(to_normal(G.lo[d][x], d), p.gamma), d);
              for (int q = 0; q < 5; ++q) dF[d][q] = fu[q] - fl[q];
            }
            for (int q = 0; q < 5; ++q) inc[x][q] = (dF[0][q] + dF[1][q]) + dF[2][q];
          }
    }
    for (int d = 0; d < 3; ++d) {
      int lo_[3], hi_[3], c[3];
      fs_lo(d, lo_, hi_);
      for (c[2] = lo_[2]; c[2] <= hi_[2]; ++c[2])
        for (c[1] = lo_[1]; c[1] <= hi_[1]; ++c[1])
          for (c[0] = lo_[0]; c[0] <= hi_[0]; ++c[0]) {
            const size_t x = G.id(c);
            for (int side = 0; side < 2; ++side) {
              std::vector<V5<R>>& fs = side ? G.up[d] : G.lo[d];
              V5<R> Uc = prim2cons(fs[x], p.gamma);
              for (int q = 0; q < 5; ++q) Uc[q] = Uc[q] - R(0.5) * nu * inc[x][q];
              fs[x] = cons2prim(Uc, p, st);
            }
          }
    }
  } else {
    // ---- VL (Falle 1991 variant; Stone & Gardiner 2009; S12) ----
    const int h = (p.recon == 0) ? 2 : 3;  // half-step state needed on [-h, 16+h)^3
    // (1) first-order fluxes from cell-centred states, same solver
    for (int d = 0; d < 3; ++d) {
      int lo_[3] = {-h, -h, -h}, hi_[3] = {PS + h - 1, PS + h - 1, PS + h - 1};
      hi_[d] = PS + h;
      flux_direction(G, G.W, G.W, G.F1[d], d, lo_, hi_, p, st);
    }
    // (2) U^{n+1/2} = U^n - nu/2 * sum_d dF1_d ; back to primitive
    G.Uh.resize(n);
    std::vector<V5<R>> Wh(n);
    {
      int c[3];
      for (c[2] = -h; c[2] < PS + h; ++c[2])
        for (c[1] = -h; c[1] < PS + h; ++c[1])
          for (c[0] = -h; c[0] < PS + h; ++c[0]) {
            const size_t x = G.id(c);
            V5<R> Uc = G.U[x];
            const int ux[3] = {c[0] + 1, c[1], c[2]}, uy[3] = {c[0], c[1] + 1, c[2]}, uz[3] = {c[0], c[1], c[2] + 1};
            for (int q = 0; q < 5; ++q)
              Uc[q] = Uc[q] - R(0.5) * nu *
                                  (((G.F1[0][G.id(ux)][q] - G.F1[0][x][q]) + (G.F1[1][G.id(uy)][q] - G.F1[1][x][q])) +
                                   (G.F1[2][G.id(uz)][q] - G.F1[2][x][q]));
            G.Uh[x] = Uc;
            Wh[x] = cons2prim(Uc, p, st);
          }
    }
    // (3) untraced reconstruction of the half-step state
    for (int d = 0; d < 3; ++d) {
      int lo_[3], hi_[3];
      fs_lo(d, lo_, hi_);
      recon_direction(G, Wh, d, lo_, hi_, p, false);
    }
  }
  // final fluxes F_d at f_d in [0,16], transverse in [0,16)   PAPER.md:41 (CTU), 40 (MHM, VL)
  for (int d = 0; d < 3; ++d) {
    int lo_[3], hi_[3];
    ff(d, lo_, hi_);
    flux_direction(G, G.up[d], G.lo[d], G.F2[d], d, lo_, hi_, p, st);
  }
  // conservative update (PAPER.md:43 step (4)); summation order S18
  const size_t ni = (size_t)PS * PS * PS;
  for (int k = 0; k < PS; ++k)
    for (int j = 0; j < PS; ++j)
      for (int i = 0; i < PS; ++i) {
        const size_t x = G.id(i, j, k), xo = ((size_t)k * PS + j) * PS + i;
        V5<R> Un;
        for (int q = 0; q < 5; ++q)
          Un[q] = G.U[x][q] - nu * (((G.F2[0][G.id(i + 1, j, k)][q] - G.F2[0][x][q]) +
                                     (G.F2[1][G.id(i, j + 1, k)][q] - G.F2[1][x][q])) +
                                    (G.F2[2][G.id(i, j, k + 1)][q] - G.F2[2][x][q]));
        const V5<R> Wn = cons2prim(Un, p, st);  // counts non-positive final states; applies floors if any
        if (p.min_dens > R(0) || p.min_pres > R(0)) Un = prim2cons(Wn, p.gamma);
        for (int q = 0; q < 5; ++q) out[(size_t)q * ni + xo] = Un[q];
      }
  // store the fluxes across patch boundaries f in {0,8,16} (PAPER.md:44 step (5); S16, S17)
  if (face_flux) {
    for (int d = 0; d < 3; ++d)
      for (int s = 0; s < 3; ++s) {
        const int f = 8 * s;
        for (int q = 0; q < 5; ++q)
          for (int b = 0; b < PS; ++b)
            for (int a = 0; a < PS; ++a) {
              // in-plane order: d=x -> [k][j], d=y -> [k][i], d=z -> [j][i] (lower axis fastest)
              int c[3];
              c[d] = f;
              c[d == 0 ? 1 : 0] = a;
              c[d == 2 ? 1 : 2] = b;
              face_flux[(((size_t)(3 * d + s) * 5 + q) * PS + b) * PS + a] = G.F2[d][G.id(c)][q];
            }
      }
  }
}

// c6. hydro_dt: maximum wave speed over the interior cells of all groups.
template <class R> R max_speed(const R* u, int Ng, int g, R gamma, int norm) {
  const int S = PS + 2 * g;
  const size_t n = (size_t)S * S * S;
  R best = R(0);
  bool bad = false;
  for (int gi = 0; gi < Ng; ++gi) {
    const R* b = u + (size_t)gi * 5 * n;
    for (int k = 0; k < PS; ++k)
      for (int j = 0; j < PS; ++j)
        for (int i = 0; i < PS; ++i) {
          const size_t x = ((size_t)(k + g) * S + (j + g)) * S + (i + g);
          const R rho = b[x], vx = b[n + x] / rho, vy = b[2 * n + x] / rho, vz = b[3 * n + x] / rho;
          const R P = (gamma - R(1)) * (b[4 * n + x] - R(0.5) * rho * ((vx * vx + vy * vy) + vz * vz));
          if (!(rho > R(0)) || !(P > R(0))) { bad = true; continue; }
          const R c = std::sqrt(gamma * P / rho);
          const R ax = std::fabs(vx), ay = std::fabs(vy), az = std::fabs(vz);
          const R s = norm == 0 ? std::max(std::max(ax, ay), az) + c : ((ax + ay) + az) + R(3) * c;
          if (!(s == s)) bad = true;
          best = std::max(best, s);
        }
  }
  return bad ? std::nan("") : best;
}

}  // namespace

// =============================================================================================
// C ABI for ctypes (tests / bench cpu_baseline only)
extern "C" {

typedef struct oracle_opts {
  int recon, nghost, char_limit;
  double minmod_coeff;
  int roe_fallback;
  double min_dens, min_pres;
  long long* status;  // host, [8] accumulated: see Status
  int nthreads;       // patch-level parallel-for over groups; 1 = single thread
} oracle_opts;

int oracle_min_ghost(int scheme, int recon) { return (scheme == 1 ? 3 : 2) + (recon == 1 ? 1 : 0); }

}  // extern "C"

namespace {
template <class R>
int solve_batch(const R* in, R* out, R* face_flux, int Ng, R dt, R dh, R gamma, int scheme, int riemann_, int limiter,
                const oracle_opts* o) {
  Params<R> p;
  p.gamma = gamma;
  p.nu = dt / dh;
  p.scheme = scheme;
  p.riemann = riemann_;
  p.limiter = limiter;
  p.recon = o ? o->recon : 0;
  p.char_limit = o ? o->char_limit : 0;
  p.roe_fallback = (o && o->roe_fallback) ? o->roe_fallback : 1;
  p.theta = (o && o->minmod_coeff > 0) ? (R)o->minmod_coeff : R(1.5);
  p.min_dens = o ? (R)o->min_dens : R(0);
  p.min_pres = o ? (R)o->min_pres : R(0);
  const int gmin = oracle_min_ghost(scheme, p.recon);
  const int g = (o && o->nghost) ? o->nghost : gmin;
  if (g < gmin || scheme < 0 || scheme > 2 || riemann_ < 0 || riemann_ > 3 || limiter < 0 || limiter > 3) return -1;
  const int S = PS + 2 * g;
  const size_t nin = (size_t)5 * S * S * S, nout = (size_t)5 * PS * PS * PS, nff = (size_t)9 * 5 * PS * PS;
  int nt = (o && o->nthreads > 0) ? o->nthreads : 1;
  Status total;
#ifdef _OPENMP
#pragma omp parallel for num_threads(nt) schedule(dynamic, 1)
#endif
  for (int gi = 0; gi < Ng; ++gi) {
    Status st;
    solve_group<R>(in + gi * nin, out + gi * nout, face_flux ? face_flux + gi * nff : nullptr, g, p, &st);
#ifdef _OPENMP
#pragma omp critical
#endif
    for (int q = 0; q < 8; ++q) total.c[q] += st.c[q];
  }
  (void)nt;
  if (o && o->status)
    for (int q = 0; q < 8; ++q) o->status[q] += total.c[q];
  return 0;
}

template <class R> Params<R> unit_params(R gamma, R nu, int riemann_, int limiter, int recon, int char_limit, R theta, int fb) {
  Params<R> p;
  p.gamma = gamma;
  p.nu = nu;
  p.scheme = 2;
  p.riemann = riemann_;
  p.limiter = limiter;
  p.recon = recon;
  p.char_limit = char_limit;
  p.roe_fallback = fb ? fb : 1;
  p.theta = theta > 0 ? theta : R(1.5);
  p.min_dens = 0;
  p.min_pres = 0;
  return p;
}
}  // namespace

extern "C" {

int oracle_hydro_solve_f64(const double* in, double* out, double* face_flux, int Ng, double dt, double dh, double gamma,
                           int scheme, int riemann_, int limiter, const oracle_opts* o) {
  return solve_batch<double>(in, out, face_flux, Ng, dt, dh, gamma, scheme, riemann_, limiter, o);
}
int oracle_hydro_solve_f32(const float* in, float* out, float* face_flux, int Ng, float dt, float dh, float gamma,
                           int scheme, int riemann_, int limiter, const oracle_opts* o) {
  return solve_batch<float>(in, out, face_flux, Ng, dt, dh, gamma, scheme, riemann_, limiter, o);
}
double oracle_hydro_dt_f64(const double* u, int Ng, int nghost, double gamma, int norm) {
  return max_speed<double>(u, Ng, nghost, gamma, norm);
}
float oracle_hydro_dt_f32(const float* u, int Ng, int nghost, float gamma, int norm) {
  return max_speed<float>(u, Ng, nghost, gamma, norm);
}

// ---- unit entry points used by the pins (normal frame: rho, vn, vt1, vt2, P) ----
// status: host long long[8] or NULL
int oracle_riemann_f64(int solver, const double* WL, const double* WR, double gamma, int roe_fallback, double* F,
                       long long* status) {
  Params<double> p = unit_params<double>(gamma, 0, solver, 1, 0, 0, 0, roe_fallback);
  Status st;
  V5<double> l, r;
  for (int q = 0; q < 5; ++q) { l[q] = WL[q]; r[q] = WR[q]; }
  const V5<double> f = riemann(l, r, p, &st, false);
  for (int q = 0; q < 5; ++q) F[q] = f[q];
  if (status) for (int q = 0; q < 8; ++q) status[q] += st.c[q];
  return 0;
}
int oracle_riemann_f32(int solver, const float* WL, const float* WR, float gamma, int roe_fallback, float* F,
                       long long* status) {
  Params<float> p = unit_params<float>(gamma, 0, solver, 1, 0, 0, 0, roe_fallback);
  Status st;
  V5<float> l, r;
  for (int q = 0; q < 5; ++q) { l[q] = WL[q]; r[q] = WR[q]; }
  const V5<float> f = riemann(l, r, p, &st, false);
  for (int q = 0; q < 5; ++q) F[q] = f[q];
  if (status) for (int q = 0; q < 8; ++q) status[q] += st.c[q];
  return 0;
}
// exact-solver star state (p*, u*) ; returns 0 ok, 1 vacuum, 2 not converged
int oracle_exact_star_f64(const double* WL, const double* WR, double gamma, double* pstar, double* ustar) {
  V5<double> l, r;
  for (int q = 0; q < 5; ++q) { l[q] = WL[q]; r[q] = WR[q]; }
  bool conv;
  if (!exact_star(l, r, gamma, *pstar, *ustar, conv)) return 1;
  return conv ? 0 : 2;
}
// exact solution sampled at x/t = 0 (primitive, normal frame)
int oracle_exact_sample0_f64(const double* WL, const double* WR, double gamma, double* W) {
  V5<double> l, r;
  for (int q = 0; q < 5; ++q) { l[q] = WL[q]; r[q] = WR[q]; }
  double ps, us;
  bool conv;
  if (!exact_star(l, r, gamma, ps, us, conv)) return 1;
  const V5<double> w = exact_sample0(l, r, gamma, ps, us);
  for (int q = 0; q < 5; ++q) W[q] = w[q];
  return conv ? 0 : 2;
}
double oracle_limited_slope_f64(double dL, double dR, int limiter, double theta) {
  return limited_slope<double>(dL, dR, 0.5 * (dL + dR), limiter, theta);
}
// face values of the middle cell of a 5-cell normal-frame pencil W5[5][5] (cells i-2..i+2)
int oracle_reconstruct_f64(const double* W5, double gamma, double nu, int recon, int limiter, int char_limit,
                           double theta, int trace, double* Wlo, double* Wup) {
  Params<double> p = unit_params<double>(gamma, nu, 3, limiter, recon, char_limit, theta, 1);
  V5<double> pencil[5], l, u;
  for (int s = 0; s < 5; ++s) for (int q = 0; q < 5; ++q) pencil[s][q] = W5[s * 5 + q];
  reconstruct(&pencil[2], p, trace != 0, l, u);
  for (int q = 0; q < 5; ++q) { Wlo[q] = l[q]; Wup[q] = u[q]; }
  return 0;
}
// eigenvector helpers for P4: a = L(W).d ; d = sum a R(W)
void oracle_eig_project_f64(const double* W, double gamma, const double* d, double* a) {
  V5<double> w, dd;
  for (int q = 0; q < 5; ++q) { w[q] = W[q]; dd[q] = d[q]; }
  const V5<double> r = eig_project(w, std::sqrt(gamma * w[4] / w[0]), dd);
  for (int q = 0; q < 5; ++q) a[q] = r[q];
}
void oracle_eig_expand_f64(const double* W, double gamma, const double* a, double* d) {
  V5<double> w, aa;
  for (int q = 0; q < 5; ++q) { w[q] = W[q]; aa[q] = a[q]; }
  const V5<double> r = eig_expand(w, std::sqrt(gamma * w[4] / w[0]), aa);
  for (int q = 0; q < 5; ++q) d[q] = r[q];
}
int oracle_max_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

}  // extern "C"
