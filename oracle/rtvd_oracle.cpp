// oracle/rtvd_oracle.cpp
//
// TEST INFRASTRUCTURE ONLY.  Plain CPU oracle of the directionally SPLIT relaxing-TVD fluid update: the
// scheme of the original GAMER ("the relaxing total variation diminishing scheme (RTVD; Jin & Xin 1995) with
// directional splitting") that the paper times next to its unsplit schemes as the memory-bound contrast.
// Only tests/ may load it; it shares no code with paper_1103_3373_b200/csrc.
//
// The paper gives no formulas.  Reading S26: the standard second-order relaxing scheme (Jin & Xin 1995) -- the
// relaxation system splits every conserved variable into a right- and a left-moving part advected with the "freezing speed"
// c, each part is advanced by a MUSCL upwind flux with the van Leer harmonic limiter, time integration is the two-stage
// (midpoint) Runge-Kutta rule.  For one sweep along direction d over a pencil of cells i, with nu = dt/dh, F_d the physical
// flux, c_i = |v_d| + sqrt(gamma P / rho) of cell i:
//     FR_i = (c_i U_i + F_d(U_i)) / 2,     FL_i = (c_i U_i - F_d(U_i)) / 2                       (right / left movers)
//     predictor   G_{i+1/2} = FR_i - FL_{i+1},        U1_i = U_i - (nu/2) (G_{i+1/2} - G_{i-1/2})
//     corrector (FR, FL re-evaluated from U1, phi(a,b) = 2ab/(a+b) if ab > 0 else 0):
//                 FR_{i+1/2} = FR_i     + phi((FR_i - FR_{i-1})/2,     (FR_{i+1} - FR_i)/2)
//                 FL_{i+1/2} = FL_{i+1} - phi((FL_{i+1} - FL_i)/2,     (FL_{i+2} - FL_{i+1})/2)
//                 H_{i+1/2}  = FR_{i+1/2} - FL_{i+1/2},     U_i <- U_i - nu (H_{i+1/2} - H_{i-1/2})
// A step is three sweeps with the same dt, in the order x, y, z (order 0) or z, y, x (order 1; alternating the two keeps
// second-order accuracy in time).  One sweep needs three ghost cells along its direction; a sweep updates the cells that are
// interior along its own direction over the transverse range later sweeps still need, so g = 3 suffices for the three sweeps.
// face_flux plane p = 3 d + s holds H of the d-sweep at the faces f = 0, 8, 16 (the flux that sweep actually used, so that
// sum(out - in) = -nu * signed boundary fluxes holds exactly as for the unsplit schemes).  No floors, no Riemann solver.
//
// Pins (tests/test_oracle_rtvd.py): uniform state bitwise; per-group flux balance and periodic conservation; mirror
// symmetry (right / left movers treated alike); total variation of an advected density profile does not grow (limiter
// sign); second-order convergence on a smooth wave (limiter corrections, midpoint rule); Sod against the exact solution.
#include <array>
#include <cmath>
#include <cstddef>
#include <vector>

namespace {
constexpr int PS = 16, GR = 3;  // ghost cells the three sweeps consume
template <class R> using V5 = std::array<R, 5>;

template <class R> struct Movers { V5<R> fr, fl; };

// right / left movers of one cell for a sweep along d (global variable order rho, mx, my, mz, E)
template <class R> Movers<R> movers(const V5<R>& U, int d, R gamma, long long* bad) {
  const R rho = U[0], vx = U[1] / rho, vy = U[2] / rho, vz = U[3] / rho;
  const R P = (gamma - R(1)) * (U[4] - R(0.5) * rho * ((vx * vx + vy * vy) + vz * vz));
  if (bad && (!(rho > R(0)) || !(P > R(0)))) ++*bad;
  const R vn = d == 0 ? vx : (d == 1 ? vy : vz);
  const R c = std::fabs(vn) + std::sqrt(gamma * P / rho);
  V5<R> F = {rho * vn, U[1] * vn, U[2] * vn, U[3] * vn, (U[4] + P) * vn};
  F[1 + d] = F[1 + d] + P;
  Movers<R> m;
  for (int q = 0; q < 5; ++q) {
    m.fr[q] = R(0.5) * (c * U[q] + F[q]);
    m.fl[q] = R(0.5) * (c * U[q] - F[q]);
  }
  return m;
}
template <class R> R phi(R a, R b) { return a * b > R(0) ? R(2) * a * b / (a + b) : R(0); }

// one sweep along a pencil u[0..n): cells 3 .. n-4 are updated; H[f] for f = 3 .. n-3 is the corrector flux at the lower face of cell f
template <class R> void sweep_pencil(std::vector<V5<R>>& u, int d, R nu, R gamma, std::vector<V5<R>>& H, long long* bad) {
  const int n = (int)u.size();
  std::vector<Movers<R>> m(n), m1(n);
  std::vector<V5<R>> u1(n);
  for (int i = 0; i < n; ++i) m[i] = movers(u[i], d, gamma, bad);
  for (int i = 1; i + 1 < n; ++i)
    for (int q = 0; q < 5; ++q) {
      const R gup = m[i].fr[q] - m[i + 1].fl[q], glo = m[i - 1].fr[q] - m[i].fl[q];
      u1[i][q] = u[i][q] - R(0.5) * nu * (gup - glo);
    }
  for (int i = 1; i + 1 < n; ++i) m1[i] = movers(u1[i], d, gamma, bad);
  H.assign(n, V5<R>{0, 0, 0, 0, 0});
  for (int f = 3; f + 2 < n; ++f)  // face between cells f-1 and f: needs movers of u1 at f-2 .. f+1
    for (int q = 0; q < 5; ++q) {
      const R frh = m1[f - 1].fr[q] + phi(R(0.5) * (m1[f - 1].fr[q] - m1[f - 2].fr[q]), R(0.5) * (m1[f].fr[q] - m1[f - 1].fr[q]));
      const R flh = m1[f].fl[q] - phi(R(0.5) * (m1[f].fl[q] - m1[f - 1].fl[q]), R(0.5) * (m1[f + 1].fl[q] - m1[f].fl[q]));
      H[f][q] = frh - flh;
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
int oracle_rtvd_solve_f64(const double* in, double* out, double* face_flux, int Ng, int g, double dt, double dh, double gamma, int order,
                          long long* status, int nthreads) {
  return solve_batch<double>(in, out, face_flux, Ng, g, dt, dh, gamma, order, status, nthreads);
}
int oracle_rtvd_solve_f32(const float* in, float* out, float* face_flux, int Ng, int g, float dt, float dh, float gamma, int order,
                          long long* status, int nthreads) {
  return solve_batch<float>(in, out, face_flux, Ng, g, dt, dh, gamma, order, status, nthreads);
}
}
