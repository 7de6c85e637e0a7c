// oracle/waf_oracle.cpp
//
// TEST INFRASTRUCTURE ONLY.  Plain CPU oracle of the directionally SPLIT weighted-average-flux update: the
// second split scheme the paper times next to its unsplit schemes ("the weighted average flux scheme (WAF; see Toro
// 2009, for an introduction)").  Only tests/ may load it; it shares no code with paper_1103_3373_b200/csrc.
//
// The paper gives no formulas.  Reading S29: the TVD version of WAF with the HLLC wave structure (Toro 2009, ch. 14.3,
// 16.4), piecewise-constant data.  One sweep along direction d over a pencil of cells, nu = dt/dh; at the face between cells L
// and R the HLLC solution (S9: Toro's pressure-based wave speeds S_L, S_R; contact speed S*) has four constant regions with
// fluxes F(1) = F_L, F(2) = F*_L, F(3) = F*_R, F(4) = F_R, F*_K = F_K + S_K (U*_K - U_K), separated by the waves k = 1, 2, 3 of
// speeds S_L, S*, S_R with Courant numbers c_k = nu S_k.  The WAF flux is
//     F = (F(1) + F(4)) / 2  -  1/2 sum_k sign(c_k) A_k (F(k+1) - F(k)),        A_k = 1 - (1 - |c_k|) B(r_k),
// B the van Leer limiter B(r) = 2r / (1 + r) for r > 0, else 0, evaluated as B(a, b) = 2a / (a + b) if a b > 0 else 0 with
// b the jump of q across wave k at this face and a the same jump at the UPWIND face (the lower face if c_k > 0, the upper one
// if c_k < 0); c_k = 0 contributes nothing.  q is the density for every component and wave, except that the two TANGENTIAL
// momentum components take, for the contact wave k = 2, their OWN jump across the contact, rho*_R v_R - rho*_L v_L (the HLLC
// solution changes a tangential velocity across the contact only -- Toro sec. 16.4 limits the shear wave on the tangential
// velocity; taking the momentum component itself keeps rho v_t consistent with rho when v_t is uniform, where a velocity jump
// of zero would switch that component alone to first order).  A = 1 is the first-order (Godunov / HLLC) flux, A = |c| Lax-Wendroff.
// Update U_i <- U_i - nu (F_{i+1/2} - F_{i-1/2}).  A step is three sweeps with the same dt in the order x, y, z (order 0) or
// z, y, x (order 1).  The scheme needs two ghost cells per sweep; the entry point works on the batches of the RTVD scheme
// (g >= 3: the 22^3 box, cells 3 .. 18 updated along the sweep over the transverse range later sweeps still need).
// face_flux plane p = 3 d + s holds the WAF flux of the d-sweep at the faces f = 0, 8, 16 (the flux that sweep used).
//
// Pins (tests/test_oracle_waf.py): uniform state bitwise; per-group flux balance; periodic conservation and mirror symmetry; a
// moving contact against the flux-limited Lax-Wendroff closed form written in NumPy (limiter, upwind choice, Courant weights);
// second-order convergence on a smooth wave (A = 1 everywhere gives rate ~1); Sod against the exact solution.
#include <array>
#include <cmath>
#include <cstddef>
#include <vector>

namespace {
constexpr int PS = 16, GR = 3;
template <class R> using V5 = std::array<R, 5>;

// HLLC solution at one face for a sweep along d: fluxes of the four regions, wave speeds, density jumps across the three waves
// and the jumps of the two tangential momentum components across the contact
template <class R> struct Face { V5<R> F[4]; R S[3]; R dq[3]; R dmt[2]; };

template <class R> struct Prim { R rho, u, vt[2], P, c, E; };
template <class R> Prim<R> prim(const V5<R>& U, int d, R gamma, long long* bad) {
  const int t1 = d == 0 ? 1 : 0, t2 = d == 2 ? 1 : 2;
  Prim<R> w;
  w.rho = U[0];
  w.u = U[1 + d] / U[0];
  w.vt[0] = U[1 + t1] / U[0];
  w.vt[1] = U[1 + t2] / U[0];
  w.E = U[4];
  w.P = (gamma - R(1)) * (U[4] - R(0.5) * U[0] * ((w.u * w.u + w.vt[0] * w.vt[0]) + w.vt[1] * w.vt[1]));
  if (bad && (!(w.rho > R(0)) || !(w.P > R(0)))) ++*bad;
  w.c = std::sqrt(gamma * w.P / w.rho);
  return w;
}
// conserved vector / physical flux in global variable order for a sweep along d
template <class R> V5<R> cons_of(R rho, R u, R v1, R v2, R E, int d) {
  const int t1 = d == 0 ? 1 : 0, t2 = d == 2 ? 1 : 2;
  V5<R> U;
  U[0] = rho; U[1 + d] = rho * u; U[1 + t1] = rho * v1; U[1 + t2] = rho * v2; U[4] = E;
  return U;
}
template <class R> V5<R> flux_of(const Prim<R>& w, int d) {
  const int t1 = d == 0 ? 1 : 0, t2 = d == 2 ? 1 : 2;
  V5<R> F;
  const R m = w.rho * w.u;
  F[0] = m; F[1 + d] = m * w.u + w.P; F[1 + t1] = m * w.vt[0]; F[1 + t2] = m * w.vt[1]; F[4] = (w.E + w.P) * w.u;
  return F;
}

template <class R> Face<R> solve_face(const Prim<R>& L, const Prim<R>& Rr, int d, R gamma) {
  Face<R> f;
  const R ppv = R(0.5) * (L.P + Rr.P) - R(0.125) * (Rr.u - L.u) * (L.rho + Rr.rho) * (L.c + Rr.c);
  const R ps = ppv > R(0) ? ppv : R(0);
  const R gf = (gamma + R(1)) / (R(2) * gamma);
  const R qL = ps <= L.P ? R(1) : std::sqrt(R(1) + gf * (ps / L.P - R(1)));
  const R qR = ps <= Rr.P ? R(1) : std::sqrt(R(1) + gf * (ps / Rr.P - R(1)));
  const R SL = L.u - L.c * qL, SR = Rr.u + Rr.c * qR;
  const R mL = L.rho * (SL - L.u), mR = Rr.rho * (SR - Rr.u);
  const R Ss = ((Rr.P - L.P) + L.u * mL - Rr.u * mR) / (mL - mR);
  f.S[0] = SL; f.S[1] = Ss; f.S[2] = SR;
  const R rsL = mL / (SL - Ss), rsR = mR / (SR - Ss);  // rho*_K
  const V5<R> UL = cons_of(L.rho, L.u, L.vt[0], L.vt[1], L.E, d), UR = cons_of(Rr.rho, Rr.u, Rr.vt[0], Rr.vt[1], Rr.E, d);
  const V5<R> UsL = cons_of(rsL, Ss, L.vt[0], L.vt[1], rsL * (L.E / L.rho + (Ss - L.u) * (Ss + L.P / mL)), d);
  const V5<R> UsR = cons_of(rsR, Ss, Rr.vt[0], Rr.vt[1], rsR * (Rr.E / Rr.rho + (Ss - Rr.u) * (Ss + Rr.P / mR)), d);
  f.F[0] = flux_of(L, d);
  f.F[3] = flux_of(Rr, d);
  for (int q = 0; q < 5; ++q) {
    f.F[1][q] = f.F[0][q] + SL * (UsL[q] - UL[q]);
    f.F[2][q] = f.F[3][q] + SR * (UsR[q] - UR[q]);
  }
  f.dq[0] = rsL - L.rho; f.dq[1] = rsR - rsL; f.dq[2] = Rr.rho - rsR;
  f.dmt[0] = rsR * Rr.vt[0] - rsL * L.vt[0]; f.dmt[1] = rsR * Rr.vt[1] - rsL * L.vt[1];
  return f;
}
template <class R> R limB(R a, R b) { return a * b > R(0) ? R(2) * a / (a + b) : R(0); }

// one sweep along a pencil u[0..n): cells 3 .. n-4 are updated; H[f] for f = 3 .. n-3 is the WAF flux at the lower face of cell f
template <class R> void sweep_pencil(std::vector<V5<R>>& u, int d, R nu, R gamma, std::vector<V5<R>>& H, long long* bad) {
  const int n = (int)u.size();
  const int t1 = d == 0 ? 1 : 0, t2 = d == 2 ? 1 : 2;
  std::vector<Prim<R>> w(n);
  for (int i = 0; i < n; ++i) w[i] = prim(u[i], d, gamma, bad);
  std::vector<Face<R>> fs(n);  // fs[f]: face between cells f-1 and f
  for (int f = 1; f < n; ++f) fs[f] = solve_face(w[f - 1], w[f], d, gamma);
  H.assign(n, V5<R>{0, 0, 0, 0, 0});
  for (int f = 3; f + 2 < n; ++f) {
    const Face<R>& c = fs[f];
    for (int q = 0; q < 5; ++q) {
      R acc = R(0.5) * (c.F[0][q] + c.F[3][q]);
      for (int k = 0; k < 3; ++k) {
        const R ck = nu * c.S[k];
        if (ck == R(0)) continue;
        const Face<R>& up = ck > R(0) ? fs[f - 1] : fs[f + 1];
        R a = up.dq[k], b = c.dq[k];
        if (k == 1 && q == 1 + t1) { a = up.dmt[0]; b = c.dmt[0]; }
        if (k == 1 && q == 1 + t2) { a = up.dmt[1]; b = c.dmt[1]; }
        const R A = R(1) - (R(1) - std::fabs(ck)) * limB(a, b);
        const R sg = ck > R(0) ? R(1) : R(-1);
        acc = acc - R(0.5) * sg * A * (c.F[k + 1][q] - c.F[k][q]);
      }
      H[f][q] = acc;
    }
  }
  for (int i = 3; i + 3 < n; ++i)
    for (int q = 0; q < 5; ++q) u[i][q] = u[i][q] - nu * (H[i + 1][q] - H[i][q]);
}

template <class R>
void solve_group(const R* in, R* out, R* face_flux, int g, R nu, R gamma, int order, long long* status) {
  const int S = PS + 2 * g, W = PS + 2 * GR, o = g - GR;
  const size_t nS = (size_t)S * S * S;
  std::vector<V5<R>> box((size_t)W * W * W);
  auto at = [&](int i, int j, int k) -> V5<R>& { return box[((size_t)(k + GR) * W + (j + GR)) * W + (i + GR)]; };
  for (int k = -GR; k < PS + GR; ++k)
    for (int j = -GR; j < PS + GR; ++j)
      for (int i = -GR; i < PS + GR; ++i)
        for (int q = 0; q < 5; ++q) at(i, j, k)[q] = in[q * nS + ((size_t)(k + GR + o) * S + (j + GR + o)) * S + (i + GR + o)];
  bool done[3] = {false, false, false};  // directions already swept: their transverse range has shrunk to the interior
  for (int s = 0; s < 3; ++s) {
    const int d = order == 0 ? s : 2 - s;
    const int t1 = d == 0 ? 1 : 0, t2 = d == 2 ? 1 : 2;
    const int lo1 = done[t1] ? 0 : -GR, hi1 = done[t1] ? PS : PS + GR, lo2 = done[t2] ? 0 : -GR, hi2 = done[t2] ? PS : PS + GR;
    for (int b = lo2; b < hi2; ++b)
      for (int a = lo1; a < hi1; ++a) {
        std::vector<V5<R>> pen(W), H;
        int c[3];
        c[t1] = a; c[t2] = b;
        for (int x = 0; x < W; ++x) { c[d] = x - GR; pen[x] = at(c[0], c[1], c[2]); }
        sweep_pencil(pen, d, nu, gamma, H, status ? status + 1 : nullptr);
        for (int x = GR; x < GR + PS; ++x) { c[d] = x - GR; at(c[0], c[1], c[2]) = pen[x]; }
        if (face_flux && a >= 0 && a < PS && b >= 0 && b < PS)
          for (int sp = 0; sp < 3; ++sp)
            for (int q = 0; q < 5; ++q) face_flux[(((size_t)(3 * d + sp) * 5 + q) * PS + b) * PS + a] = H[GR + 8 * sp][q];
      }
    done[d] = true;
  }
  const size_t ni = (size_t)PS * PS * PS;
  for (int k = 0; k < PS; ++k)
    for (int j = 0; j < PS; ++j)
      for (int i = 0; i < PS; ++i)
        for (int q = 0; q < 5; ++q) out[q * ni + ((size_t)k * PS + j) * PS + i] = at(i, j, k)[q];
}

template <class R>
int solve_batch(const R* in, R* out, R* face_flux, int Ng, int g, R dt, R dh, R gamma, int order, long long* status, int nthreads) {
  if (g < GR || Ng < 0 || order < 0 || order > 1) return -1;
  const int S = PS + 2 * g;
  const size_t in_n = (size_t)5 * S * S * S, out_n = (size_t)5 * PS * PS * PS, ff_n = (size_t)9 * 5 * PS * PS;
  long long tot[2] = {0, 0};
#pragma omp parallel for num_threads(nthreads > 0 ? nthreads : 1) schedule(dynamic)
  for (int n = 0; n < Ng; ++n) {
    long long st[2] = {0, 0};
    solve_group<R>(in + n * in_n, out + n * out_n, face_flux ? face_flux + n * ff_n : nullptr, g, dt / dh, gamma, order, st);
#pragma omp atomic
    tot[1] += st[1];
  }
  if (status) status[1] += tot[1];
  return 0;
}
}  // namespace

extern "C" {
int oracle_waf_solve_f64(const double* in, double* out, double* face_flux, int Ng, int g, double dt, double dh, double gamma, int order,
                         long long* status, int nthreads) {
  return solve_batch<double>(in, out, face_flux, Ng, g, dt, dh, gamma, order, status, nthreads);
}
int oracle_waf_solve_f32(const float* in, float* out, float* face_flux, int Ng, int g, float dt, float dh, float gamma, int order,
                         long long* status, int nthreads) {
  return solve_batch<float>(in, out, face_flux, Ng, g, dt, dh, gamma, order, status, nthreads);
}
}
