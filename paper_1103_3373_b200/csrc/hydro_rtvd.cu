// hydro_rtvd.cu -- the directionally SPLIT relaxing-TVD update of a batch of patch groups: the scheme of
// the original GAMER (Jin & Xin 1995) that the paper times next to its unsplit schemes as the contrast with low
// arithmetic intensity ("for the directionally split schemes ... the integration only requires 1D stencils").
// Reading S26 of DESIGN.md (formulas in oracle/rtvd_oracle.cpp's header, restated here independently): every conserved variable
// is split into a right- and a left-moving part advected with the freezing speed c = |v_d| + c_s; midpoint Runge-Kutta with a
// first-order predictor and a van-Leer-limited MUSCL corrector; three sweeps per step, x,y,z (order 0) or z,y,x (order 1).
//
// Organisation: persistent CTAs, one patch group at a time; a thread owns one pencil of a sweep and marches along it with a
// register window (two limiter stencils of movers, the predictor flux, the last corrector flux), so that every cell's movers
// are evaluated once.  Sweep 1 reads `in`, sweep 3 writes `out`; the two intermediate boxes (only the range later sweeps still
// need: 22x22x16 and 22x16x16 cells) live in a caller-supplied scratch slot per CTA that stays L2-resident.  ~110 flops against
// ~85 bytes of HBM traffic per cell update: HBM-bound, unlike the Riemann-solver schemes.  Part of the CUDA product path.
#include <cuda_runtime.h>
#include <cstdint>

#include "../../include/hydro.h"
#include "hydro_math.cuh"
#include "hydro_ptx.cuh"

namespace hydro {

constexpr int RT_G = 3, RT_W = PS + 2 * RT_G, RT_NT = 256;

template <class R> struct Mv { V5<R> fr, fl; };
// right / left movers of one cell for a sweep along D: (c U +- F_D(U)) / 2
template <int D, class R> __device__ __forceinline__ Mv<R> rt_movers(const V5<R>& U, R gamma, int& bad) {
  const R ir = m_rcp(U[0]);
  const R vx = U[1] * ir, vy = U[2] * ir, vz = U[3] * ir;
  const R P = (gamma - R(1)) * (U[4] - R(0.5) * U[0] * ((vx * vx + vy * vy) + vz * vz));
  bad += (U[0] > R(0) && P > R(0)) ? 0 : 1;
  const R vn = D == 0 ? vx : (D == 1 ? vy : vz);
  const R c = m_abs(vn) + m_sqrt(gamma * P * ir);
  V5<R> F;
  F[0] = U[0] * vn; F[1] = U[1] * vn; F[2] = U[2] * vn; F[3] = U[3] * vn; F[4] = (U[4] + P) * vn;
  F[1 + D] = F[1 + D] + P;
  Mv<R> m;
#pragma unroll
  for (int q = 0; q < 5; ++q) {
    m.fr[q] = R(0.5) * (c * U[q] + F[q]);
    m.fl[q] = R(0.5) * (c * U[q] - F[q]);
  }
  return m;
}
template <class R> __device__ __forceinline__ R rt_phi(R a, R b) {
  const R p = a * b;
  return p > R(0) ? m_div(p + p, a + b) : R(0);
}
// phi(a/2, b/2) = a b / (a + b): the halves of the limiter's arguments and the factor two cancel exactly in binary arithmetic,
// three instructions fewer per limiter evaluation (ten evaluations per cell and sweep)
template <class R> __device__ __forceinline__ R rt_phi_half(R a, R b) {
  const R p = a * b;
  return p > R(0) ? m_div(p, a + b) : R(0);
}

// One sweep along D of the pencils (a, b), a in [0, na), b in [0, nb).  src cell (q, a, b, x) at src[q sq + a sa + b sb + x sx],
// x = 0 .. 21; dst likewise for the 16 updated cells x - 3.  ff: plane base of direction D (3 planes x 5 x 256) or nullptr;
// (a - fa0, b - fb0) are the in-plane interior coordinates of the pencil (lower axis fastest).
// The march is unrolled by six -- the period of its register windows (three cells of right movers, three of left movers, two
// predictor / corrector fluxes) -- so that the windows rotate by renaming, not by moves (the rolled loop spent 29 % of its
// instructions on MOV), and the next cell's five loads are issued before the current cell's arithmetic.
template <int D, class R, int NT = RT_NT>
__device__ __forceinline__ void rt_sweep(const R* __restrict__ src, size_t sq, int sa, int sb, int sx, R* __restrict__ dst, size_t dq,
                                         int da, int db, int dx, int na, int nb, int fa0, int fb0, R* __restrict__ ff, R nu, R gamma,
                                         int& bad) {
  for (int pidx = threadIdx.x; pidx < na * nb; pidx += NT) {
    const int b = pidx / na, a = pidx - b * na;
    const R* s = src + (size_t)a * sa + (size_t)b * sb;
    R* d = dst + (size_t)a * da + (size_t)b * db;
    const int ta = a - fa0, tb = b - fb0;
    R* fp = (ff && ta >= 0 && ta < PS && tb >= 0 && tb < PS) ? ff + tb * PS + ta : nullptr;
    V5<R> Uw[2], frw[2], Gw[2], Hw[2];  // U, right movers of U, predictor flux, corrector flux: current and previous
    V5<R> r1[3], l1[3];                 // right / left movers of the predicted state u1, cells x-1, x-2, x-3 (slot = cell % 3)
    V5<R> Unext;
#pragma unroll
    for (int q = 0; q < 5; ++q) {
      Uw[0][q] = Uw[1][q] = frw[0][q] = frw[1][q] = Gw[0][q] = Gw[1][q] = Hw[0][q] = Hw[1][q] = R(0);
      r1[0][q] = r1[1][q] = r1[2][q] = l1[0][q] = l1[1][q] = l1[2][q] = R(0);
      Unext[q] = s[q * sq];
    }
#pragma unroll 1
    for (int x0 = 0; x0 < RT_W; x0 += 6) {
#pragma unroll
      for (int u = 0; u < 6; ++u) {
        const int x = x0 + u;
        if (x < RT_W) {
          V5<R>& U = Uw[u & 1];
          const V5<R>& Uprev = Uw[(u + 1) & 1];
          U = Unext;
          if (x + 1 < RT_W) {
#pragma unroll
            for (int q = 0; q < 5; ++q) Unext[q] = s[q * sq + (size_t)(x + 1) * sx];
          }
          const Mv<R> m = rt_movers<D>(U, gamma, bad);
          if (x >= 1) {
            V5<R>& G = Gw[u & 1];  // predictor flux at the face between x-1 and x
            const V5<R>& Glo = Gw[(u + 1) & 1];
#pragma unroll
            for (int q = 0; q < 5; ++q) G[q] = frw[(u + 1) & 1][q] - m.fl[q];
            if (x >= 2) {  // u1 of cell x-1, its movers, the corrector flux at the lower face of cell x-2, the update of cell x-3
              V5<R> u1;
#pragma unroll
              for (int q = 0; q < 5; ++q) u1[q] = Uprev[q] - R(0.5) * nu * (G[q] - Glo[q]);
              const Mv<R> m1 = rt_movers<D>(u1, gamma, bad);  // cell x-1 -> slot (u + 5) % 3
              constexpr int dummy = 0; (void)dummy;
              const int c1 = (u + 5) % 3, c2 = (u + 4) % 3, c3 = (u + 3) % 3;  // slots of cells x-1, x-2, x-3 (compile time: u is)
              V5<R> fr4 = r1[c1];  // right movers of cell x-4 still sit in the slot cell x-1 takes
              r1[c1] = m1.fr;
              l1[c1] = m1.fl;
              if (x >= 5) {  // face f = x-2: right movers of cells x-4, x-3, x-2; left movers of cells x-3, x-2, x-1
                V5<R>& H = Hw[u & 1];
                const V5<R>& Hlo = Hw[(u + 1) & 1];
#pragma unroll
                for (int q = 0; q < 5; ++q) {
                  const R frh = r1[c3][q] + rt_phi_half(r1[c3][q] - fr4[q], r1[c2][q] - r1[c3][q]);
                  const R flh = l1[c2][q] - rt_phi_half(l1[c2][q] - l1[c3][q], l1[c1][q] - l1[c2][q]);
                  H[q] = frh - flh;
                }
                const int f = x - 2 - RT_G;  // face index of the group: 0 .. 16
                if (fp && (f & 7) == 0) {
#pragma unroll
                  for (int q = 0; q < 5; ++q) fp[((f >> 3) * 5 + q) * (PS * PS)] = H[q];
                }
                if (x >= 6) {  // cell x-3 = interior cell f-1; U[x-3] is re-read (an L1 hit) rather than carried through the window
#pragma unroll
                  for (int q = 0; q < 5; ++q)
                    d[q * dq + (size_t)(x - 3 - RT_G) * dx] = s[q * sq + (size_t)(x - 3) * sx] - nu * (H[q] - Hlo[q]);
                }
              }
            }
          }
          frw[u & 1] = m.fr;
        }
      }
    }
  }
}

// ---- the split WEIGHTED AVERAGE FLUX scheme ("WAF; see Toro 2009"): reading S29 of DESIGN.md, restated here
// independently of oracle/waf_oracle.cpp.  TVD WAF with the HLLC wave structure on piecewise-constant data: at a face the
// HLLC solution has regions F(1..4) = F_L, F*_L, F*_R, F_R separated by the waves S_L, S*, S_R (S9: Toro's pressure-based
// speeds); F = (F(1) + F(4))/2 - 1/2 sum_k sign(c_k) A_k (F(k+1) - F(k)), c_k = nu S_k, A_k = 1 - (1 - |c_k|) B(a, b), B the
// van Leer limiter 2a/(a+b) for ab > 0 (else 0) of the jump b of q across wave k at this face and the jump a at the upwind
// face; q = rho, except that the tangential momentum components take their own jump across the contact for k = 2.
// Everything below works in the NORMAL frame of the sweep: (rho, m_n, m_t1, m_t2, E).
template <class R> struct WCell { R rho, u, v1, v2, P, c, E; };
template <class R> struct WJump { R q[3], t1, t2; };                 // jumps across the three waves; tangential momenta across the contact
template <class R> struct WWave { R SL, Ss, SR, rsL, rsR; };           // wave speeds and star densities of one face
template <class R> __device__ __forceinline__ WCell<R> waf_cell(const V5<R>& U, R gamma, int& bad) {
  WCell<R> w;
  const R ir = m_rcp(U[0]);
  w.rho = U[0]; w.u = U[1] * ir; w.v1 = U[2] * ir; w.v2 = U[3] * ir; w.E = U[4];
  w.P = (gamma - R(1)) * (U[4] - R(0.5) * U[0] * ((w.u * w.u + w.v1 * w.v1) + w.v2 * w.v2));
  bad += (w.rho > R(0) && w.P > R(0)) ? 0 : 1;
  w.c = m_sqrt(gamma * w.P * ir);
  return w;
}
// first half of a face: the wave structure and the jumps the limiter looks at (the neighbouring faces need these, not the fluxes)
template <class R> __device__ __forceinline__ void waf_waves(const WCell<R>& L, const WCell<R>& Rr, R gamma, WWave<R>& w, WJump<R>& j) {
  const R ppv = R(0.5) * (L.P + Rr.P) - R(0.125) * (Rr.u - L.u) * (L.rho + Rr.rho) * (L.c + Rr.c);
  const R ps = m_max(ppv, R(0));
  const R gf = (gamma + R(1)) * m_rcp(gamma + gamma);
  const R qL = ps <= L.P ? R(1) : m_sqrt(R(1) + gf * (m_div(ps, L.P) - R(1)));
  const R qR = ps <= Rr.P ? R(1) : m_sqrt(R(1) + gf * (m_div(ps, Rr.P) - R(1)));
  w.SL = L.u - L.c * qL;
  w.SR = Rr.u + Rr.c * qR;
  const R mL = L.rho * (w.SL - L.u), mR = Rr.rho * (w.SR - Rr.u);
  w.Ss = m_div((Rr.P - L.P) + L.u * mL - Rr.u * mR, mL - mR);
  w.rsL = m_div(mL, w.SL - w.Ss);
  w.rsR = m_div(mR, w.SR - w.Ss);
  j.q[0] = w.rsL - L.rho; j.q[1] = w.rsR - w.rsL; j.q[2] = Rr.rho - w.rsR;
  j.t1 = w.rsR * Rr.v1 - w.rsL * L.v1;
  j.t2 = w.rsR * Rr.v2 - w.rsL * L.v2;
}
template <class R> __device__ __forceinline__ R waf_B(R a, R b) { return a * b > R(0) ? m_div(a + a, a + b) : R(0); }
// half the signed weight sign(c) A / 2 of one wave for one limiter pair
template <class R> __device__ __forceinline__ R waf_w(R c, R a, R b) {
  const R sg = c > R(0) ? R(0.5) : (c < R(0) ? R(-0.5) : R(0));
  return sg * (R(1) - (R(1) - m_abs(c)) * waf_B(a, b));
}
// second half: the WAF flux of the face (normal frame) from its cells, its waves, its own jumps jc and those of the lower (jl)
// and upper (ju) faces.  The region fluxes are formed here and consumed at once, so that only the wave data of a face is carried
// from step to step of the march
template <class R> __device__ __forceinline__ V5<R> waf_flux(const WCell<R>& L, const WCell<R>& Rr, const WWave<R>& w, R nu,
                                                             const WJump<R>& jl, const WJump<R>& jc, const WJump<R>& ju) {
  const R mL = L.rho * (w.SL - L.u), mR = Rr.rho * (w.SR - Rr.u);
  const R EsL = w.rsL * (m_div(L.E, L.rho) + (w.Ss - L.u) * (w.Ss + m_div(L.P, mL)));
  const R EsR = w.rsR * (m_div(Rr.E, Rr.rho) + (w.Ss - Rr.u) * (w.Ss + m_div(Rr.P, mR)));
  const R mnL = L.rho * L.u, mnR = Rr.rho * Rr.u;
  V5<R> d1, d3, FL, FR;  // F*_L - F_L = S_L (U*_L - U_L);  F_R - F*_R = -S_R (U*_R - U_R);  the contact takes the rest of F_R - F_L
  d1[0] = w.SL * (w.rsL - L.rho);                  d3[0] = -w.SR * (w.rsR - Rr.rho);
  d1[1] = w.SL * (w.rsL * w.Ss - mnL);             d3[1] = -w.SR * (w.rsR * w.Ss - mnR);
  d1[2] = w.SL * (w.rsL * L.v1 - L.rho * L.v1);    d3[2] = -w.SR * (w.rsR * Rr.v1 - Rr.rho * Rr.v1);
  d1[3] = w.SL * (w.rsL * L.v2 - L.rho * L.v2);    d3[3] = -w.SR * (w.rsR * Rr.v2 - Rr.rho * Rr.v2);
  d1[4] = w.SL * (EsL - L.E);                      d3[4] = -w.SR * (EsR - Rr.E);
  FL[0] = mnL; FL[1] = mnL * L.u + L.P; FL[2] = mnL * L.v1; FL[3] = mnL * L.v2; FL[4] = (L.E + L.P) * L.u;
  FR[0] = mnR; FR[1] = mnR * Rr.u + Rr.P; FR[2] = mnR * Rr.v1; FR[3] = mnR * Rr.v2; FR[4] = (Rr.E + Rr.P) * Rr.u;
  const R c0 = nu * w.SL, c1 = nu * w.Ss, c2 = nu * w.SR;
  // upwind jumps of the three waves (selected by value: a run-time choice between two structs would put them in local memory)
  const bool p0 = c0 > R(0), p1 = c1 > R(0), p2 = c2 > R(0);
  const R w0 = waf_w(c0, p0 ? jl.q[0] : ju.q[0], jc.q[0]), w2 = waf_w(c2, p2 ? jl.q[2] : ju.q[2], jc.q[2]);
  const R w1 = waf_w(c1, p1 ? jl.q[1] : ju.q[1], jc.q[1]);
  const R w1a = waf_w(c1, p1 ? jl.t1 : ju.t1, jc.t1), w1b = waf_w(c1, p1 ? jl.t2 : ju.t2, jc.t2);
  const R wk[5] = {w1, w1, w1a, w1b, w1};
  V5<R> H;
#pragma unroll
  for (int q = 0; q < 5; ++q) {
    const R d2 = ((FR[q] - FL[q]) - d1[q]) - d3[q];
    H[q] = ((R(0.5) * (FL[q] + FR[q]) - w0 * d1[q]) - wk[q] * d2) - w2 * d3[q];
  }
  return H;
}

// One WAF sweep along D: same pencil geometry and arguments as rt_sweep (cells 3 .. 18 of the 22-cell pencil are updated, the
// scheme itself needs two of the three ghost cells).  Register windows: the cells x-2, x-1, x (primitives), the wave data of the
// faces x-1, x, the jumps of the faces x-2, x-1, x, the fluxes of the faces x-2, x-1; unrolled by their common period six.
template <int D, class R, int NT = RT_NT>
__device__ __forceinline__ void waf_sweep(const R* __restrict__ src, size_t sq, int sa, int sb, int sx, R* __restrict__ dst, size_t dq,
                                          int da, int db, int dx, int na, int nb, int fa0, int fb0, R* __restrict__ ff, R nu, R gamma,
                                          int& bad) {
  constexpr int QN = 1 + D, QT1 = D == 0 ? 2 : 1, QT2 = D == 2 ? 2 : 3;  // global indices of m_n, m_t1, m_t2
  for (int pidx = threadIdx.x; pidx < na * nb; pidx += NT) {
    const int b = pidx / na, a = pidx - b * na;
    const R* s = src + (size_t)a * sa + (size_t)b * sb;
    R* d = dst + (size_t)a * da + (size_t)b * db;
    const int ta = a - fa0, tb = b - fb0;
    R* fp = (ff && ta >= 0 && ta < PS && tb >= 0 && tb < PS) ? ff + tb * PS + ta : nullptr;
    WCell<R> cw[3];
    WWave<R> ww[2];
    WJump<R> jw[3];
    V5<R> Hw[2], Unext;
#pragma unroll
    for (int q = 0; q < 5; ++q) { Hw[0][q] = Hw[1][q] = R(0); Unext[q] = s[q * sq]; }
#pragma unroll 1
    for (int x0 = 0; x0 < RT_W; x0 += 6) {
#pragma unroll
      for (int u = 0; u < 6; ++u) {
        const int x = x0 + u;
        if (x < RT_W) {
          V5<R> Un;  // normal frame
          Un[0] = Unext[0]; Un[1] = Unext[QN]; Un[2] = Unext[QT1]; Un[3] = Unext[QT2]; Un[4] = Unext[4];
          if (x + 1 < RT_W) {
#pragma unroll
            for (int q = 0; q < 5; ++q) Unext[q] = s[q * sq + (size_t)(x + 1) * sx];
          }
          cw[u % 3] = waf_cell(Un, gamma, bad);
          if (x >= 1) waf_waves(cw[(u + 2) % 3], cw[u % 3], gamma, ww[u & 1], jw[u % 3]);  // face x, between cells x-1 and x
          if (x >= 4 && x <= RT_W - 2) {  // flux of face f = x-1 in 3 .. 19 (cells x-2, x-1): jumps of the faces x-2, x-1, x
            const V5<R> Hn = waf_flux(cw[(u + 1) % 3], cw[(u + 2) % 3], ww[(u + 1) & 1], nu, jw[(u + 1) % 3], jw[(u + 2) % 3], jw[u % 3]);
            V5<R>& H = Hw[u & 1];
            H[0] = Hn[0]; H[QN] = Hn[1]; H[QT1] = Hn[2]; H[QT2] = Hn[3]; H[4] = Hn[4];
            const int f = x - 1 - RT_G;  // face index of the group: 0 .. 16
            if (fp && (f & 7) == 0) {
#pragma unroll
              for (int q = 0; q < 5; ++q) fp[((f >> 3) * 5 + q) * (PS * PS)] = H[q];
            }
            if (x >= 5) {  // cell x-2 = interior cell f-1
              const V5<R>& Hlo = Hw[(u + 1) & 1];
#pragma unroll
              for (int q = 0; q < 5; ++q)
                d[q * dq + (size_t)(x - 2 - RT_G) * dx] = s[q * sq + (size_t)(x - 2) * sx] - nu * (H[q] - Hlo[q]);
            }
          }
        }
      }
    }
  }
}

constexpr int SPLIT_RTVD = 0, SPLIT_WAF = 1;
template <int SCHEME, int D, class R, int NT = RT_NT>
__device__ __forceinline__ void split_sweep(const R* __restrict__ src, size_t sq, int sa, int sb, int sx, R* __restrict__ dst, size_t dq,
                                            int da, int db, int dx, int na, int nb, int fa0, int fb0, R* __restrict__ ff, R nu, R gamma,
                                            int& bad) {
  if (SCHEME == SPLIT_WAF) waf_sweep<D, R, NT>(src, sq, sa, sb, sx, dst, dq, da, db, dx, na, nb, fa0, fb0, ff, nu, gamma, bad);
  else rt_sweep<D, R, NT>(src, sq, sa, sb, sx, dst, dq, da, db, dx, na, nb, fa0, fb0, ff, nu, gamma, bad);
}

template <class R, int SCHEME>
__global__ void __launch_bounds__(RT_NT, sizeof(R) == 4 ? 2 : 1)
rtvd_kernel(const R* __restrict__ in, R* __restrict__ out, R* __restrict__ face_flux, int Ng, int g, R nu_arg, R gamma, int order,
            const R* __restrict__ max_speed, R cfl, R* __restrict__ scratch, long long* status) {
  R nu = nu_arg;
  if (max_speed) nu = m_div(cfl, __ldg(max_speed));
  const int S = PS + 2 * g, o = g - RT_G;
  const size_t nS = (size_t)S * S * S;
  constexpr size_t N1 = (size_t)RT_W * RT_W * PS, N2 = (size_t)RT_W * PS * PS, NI = (size_t)PS * PS * PS;
  R* s1 = scratch + (size_t)blockIdx.x * 5 * (N1 + N2);
  R* s2 = s1 + 5 * N1;
  int bad = 0;
  for (int grp = blockIdx.x; grp < Ng; grp += gridDim.x) {
    const R* gin = in + (size_t)grp * 5 * nS + ((size_t)o * S + o) * S + o;  // first cell of the 22^3 work box
    R* gout = out + (size_t)grp * 5 * NI;
    R* gff = face_flux ? face_flux + (size_t)grp * 9 * 5 * PS * PS : nullptr;
    if (order == 0) {
      // x: pencils (j, k) of the padded box -> s1[q][k 22][j 22][i 16];  y: pencils (i, k) -> s2[q][k 22][j 16][i 16];  z: (i, j) -> out
      split_sweep<SCHEME, 0, R>(gin, nS, S, S * S, 1, s1, N1, PS, RT_W * PS, 1, RT_W, RT_W, RT_G, RT_G, gff, nu, gamma, bad);
      __syncthreads();
      split_sweep<SCHEME, 1, R>(s1, N1, 1, RT_W * PS, PS, s2, N2, 1, PS * PS, PS, PS, RT_W, 0, RT_G, gff ? gff + 3 * 5 * PS * PS : nullptr, nu, gamma, bad);
      __syncthreads();
      split_sweep<SCHEME, 2, R>(s2, N2, 1, PS, PS * PS, gout, NI, 1, PS, PS * PS, PS, PS, 0, 0, gff ? gff + 6 * 5 * PS * PS : nullptr, nu, gamma, bad);
    } else {
      // z: pencils (i, j) of the padded box -> s1[q][k 16][j 22][i 22];  y: pencils (i, k) -> s2[q][k 16][j 16][i 22];  x: (j, k) -> out
      split_sweep<SCHEME, 2, R>(gin, nS, 1, S, S * S, s1, N1, 1, RT_W, RT_W * RT_W, RT_W, RT_W, RT_G, RT_G, gff ? gff + 6 * 5 * PS * PS : nullptr, nu, gamma, bad);
      __syncthreads();
      split_sweep<SCHEME, 1, R>(s1, N1, 1, RT_W * RT_W, RT_W, s2, N2, 1, PS * RT_W, RT_W, RT_W, PS, RT_G, 0, gff ? gff + 3 * 5 * PS * PS : nullptr, nu, gamma, bad);
      __syncthreads();
      split_sweep<SCHEME, 0, R>(s2, N2, RT_W, PS * RT_W, 1, gout, NI, PS, PS * PS, 1, PS, PS, 0, 0, gff, nu, gamma, bad);
    }
    __syncthreads();  // the next group overwrites s1 / s2
  }
  if (status) {
#pragma unroll
    for (int ofs = 16; ofs > 0; ofs >>= 1) bad += __shfl_xor_sync(0xffffffffu, bad, ofs);
    if ((threadIdx.x & 31) == 0 && bad) atomicAdd(reinterpret_cast<unsigned long long*>(status + 1), (unsigned long long)bad);
  }
}

// ---- fp32, g = 3: the whole padded group (5 x 22^3 floats = 213 KB) lives in SHARED memory.  One CTA of 512 threads per SM
// loads it with five bulk async copies (a variable of a g = 3 group is one contiguous 42 592-byte piece), runs the three sweeps
// IN PLACE (a pencil belongs to one thread, and the march overwrites a cell only after its last read), and the third sweep
// writes `out`: no scratch, no intermediate traffic, no long-scoreboard stalls on L2 (the scratch kernel above spends 3.2 of its
// 6.9 stall cycles per instruction there).  The x sweep reads with a stride of 22 floats between lanes: two-way bank conflicts.
constexpr int RT_SNT = 512;
#ifndef WAF_SNT
#define WAF_SNT 256
#endif
constexpr size_t RT_SMEM = 64 + 5 * (size_t)RT_W * RT_W * RT_W * sizeof(float);
template <int SCHEME, int SNT>
__global__ void __launch_bounds__(SNT, 1)
rtvd_smem_kernel(const float* __restrict__ in, float* __restrict__ out, float* __restrict__ face_flux, int Ng, float nu_arg, float gamma,
                 int order, const float* __restrict__ max_speed, float cfl, long long* status) {
  using R = float;
  extern __shared__ __align__(16) unsigned char rt_smem[];
  uint64_t* bar = reinterpret_cast<uint64_t*>(rt_smem);
  R* box = reinterpret_cast<R*>(rt_smem + 64);  // [5][22][22][22]
  constexpr int W = RT_W, W2 = W * W, W3 = W2 * W;
  constexpr size_t NI = (size_t)PS * PS * PS;
  R nu = nu_arg;
  if (max_speed) nu = m_div(cfl, __ldg(max_speed));
  if (threadIdx.x == 0) {
    mbar_init(bar, 1);
    fence_mbar_init();
    fence_async_smem();
  }
  __syncthreads();
  int bad = 0;
  uint32_t phase = 0;
  for (int grp = blockIdx.x; grp < Ng; grp += gridDim.x) {
    if (threadIdx.x == 0) {
      fence_async_smem();  // the sweeps of the previous group wrote the box through the generic proxy
      mbar_expect_tx(bar, (uint32_t)(5 * W3 * sizeof(R)));
      const R* src = in + (size_t)grp * 5 * W3;
#pragma unroll
      for (int q = 0; q < 5; ++q) bulk_g2s(box + q * W3, src + (size_t)q * W3, (uint32_t)(W3 * sizeof(R)), bar);
    }
    mbar_wait(bar, phase);
    phase ^= 1u;
    R* gout = out + (size_t)grp * 5 * NI;
    R* gff = face_flux ? face_flux + (size_t)grp * 9 * 5 * PS * PS : nullptr;
    R* fx = gff, *fy = gff ? gff + 3 * 5 * PS * PS : nullptr, *fz = gff ? gff + 6 * 5 * PS * PS : nullptr;
    if (order == 0) {
      // x: pencils (j, k) of the box, in place;  y: pencils (i interior, k);  z: pencils (i, j) interior -> out
      split_sweep<SCHEME, 0, R, SNT>(box, W3, W, W2, 1, box + RT_G, W3, W, W2, 1, W, W, RT_G, RT_G, fx, nu, gamma, bad);
      __syncthreads();
      split_sweep<SCHEME, 1, R, SNT>(box + RT_G, W3, 1, W2, W, box + RT_G + RT_G * W, W3, 1, W2, W, PS, W, 0, RT_G, fy, nu, gamma, bad);
      __syncthreads();
      split_sweep<SCHEME, 2, R, SNT>(box + RT_G + RT_G * W, W3, 1, W, W2, gout, NI, 1, PS, PS * PS, PS, PS, 0, 0, fz, nu, gamma, bad);
    } else {
      // z: pencils (i, j) of the box, in place;  y: pencils (i, k interior);  x: pencils (j, k) interior -> out
      split_sweep<SCHEME, 2, R, SNT>(box, W3, 1, W, W2, box + RT_G * W2, W3, 1, W, W2, W, W, RT_G, RT_G, fz, nu, gamma, bad);
      __syncthreads();
      split_sweep<SCHEME, 1, R, SNT>(box + RT_G * W2, W3, 1, W2, W, box + RT_G * W2 + RT_G * W, W3, 1, W2, W, W, PS, RT_G, 0, fy, nu, gamma, bad);
      __syncthreads();
      // the x sweep comes last here: written straight to `out` its lanes (pencils j) would store 64 bytes apart, so it also runs
      // in place and the interior leaves the box in a coalesced copy
      split_sweep<SCHEME, 0, R, SNT>(box + RT_G * W2 + RT_G * W, W3, W, W2, 1, box + RT_G * W2 + RT_G * W + RT_G, W3, W, W2, 1, PS, PS, 0, 0, fx, nu, gamma, bad);
      __syncthreads();
      for (int idx = threadIdx.x; idx < 5 * (int)NI; idx += SNT) {
        const int q = idx >> 12, c = idx & 4095, k = c >> 8, j = (c >> 4) & 15, i = c & 15;
        gout[idx] = box[q * W3 + (k + RT_G) * W2 + (j + RT_G) * W + (i + RT_G)];
      }
    }
    __syncthreads();  // the next group's copies overwrite the box
  }
  if (status) {
#pragma unroll
    for (int ofs = 16; ofs > 0; ofs >>= 1) bad += __shfl_xor_sync(0xffffffffu, bad, ofs);
    if ((threadIdx.x & 31) == 0 && bad) atomicAdd(reinterpret_cast<unsigned long long*>(status + 1), (unsigned long long)bad);
  }
}

constexpr int RT_MAX_SLOTS = 148 * 2;  // 296 slots x 267 KB (fp32) stay in the 126 MB L2; 592 spilled 1.2 GB of scratch writes to HBM
inline size_t rtvd_slot_bytes(size_t elem) { return 5 * ((size_t)RT_W * RT_W * PS + (size_t)RT_W * PS * PS) * elem; }

template <class R>
static int rtvd_impl(const R* in, R* out, R* ff, int Ng, R dt, R dh, R gamma, int order, const hydro_opts* o, cudaStream_t st,
                     int scheme = SPLIT_RTVD) {
  if (Ng < 0) return HYDRO_E_COUNT;
  if (order < 0 || order > 1) return HYDRO_E_ENUM;
  const int g = (o && o->nghost) ? o->nghost : RT_G;
  if (g < RT_G || g > 8) return HYDRO_E_GHOST;
  const bool device_dt = o && o->max_speed;
  if (!(gamma > R(1)) || !(dh > R(0)) || (!device_dt && !(dt >= R(0))) || (device_dt && !(o->cfl > 0.0))) return HYDRO_E_VALUE;
  if (Ng == 0) return HYDRO_OK;
  if (!in || !out) return HYDRO_E_NULL;
  if (((uintptr_t)in & 15) || ((uintptr_t)out & 15) || ((uintptr_t)ff & 15)) return HYDRO_E_ALIGN;
  if constexpr (sizeof(R) == 4) {
    if (g == RT_G) {  // the group fits in shared memory: no scratch
      static int sms = 0;
      if (!sms) {
        int dev = 0;
        cudaGetDevice(&dev);
        if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms <= 0) sms = 148;
      }
      // RTVD: 512 threads (one pass over the 484 pencils of the first sweep, 124 registers).  WAF holds more per pencil: WAF_SNT
      // threads leave it the registers it needs
      auto kern = scheme == SPLIT_WAF ? rtvd_smem_kernel<SPLIT_WAF, WAF_SNT> : rtvd_smem_kernel<SPLIT_RTVD, RT_SNT>;
      const int nt = scheme == SPLIT_WAF ? WAF_SNT : RT_SNT;
      cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)RT_SMEM);
      if (e != cudaSuccess) return (int)e;
      kern<<<(unsigned)(Ng < sms ? Ng : sms), nt, RT_SMEM, st>>>(in, out, ff, Ng, device_dt ? 0.f : dt / dh, gamma, order,
                                                                 device_dt ? static_cast<const float*>(o->max_speed) : nullptr,
                                                                 device_dt ? (float)o->cfl : 0.f, o ? o->status : nullptr);
      return (int)cudaGetLastError();
    }
  }
  const size_t slot = rtvd_slot_bytes(sizeof(R));
  if (!o || !o->workspace || ((uintptr_t)o->workspace & 15) || o->workspace_bytes < slot) return HYDRO_E_WORKSPACE;
  long long slots = (long long)(o->workspace_bytes / slot);
  if (slots > RT_MAX_SLOTS) slots = RT_MAX_SLOTS;
  if (slots > Ng) slots = Ng;
  auto kern = scheme == SPLIT_WAF ? rtvd_kernel<R, SPLIT_WAF> : rtvd_kernel<R, SPLIT_RTVD>;
  kern<<<(unsigned)slots, RT_NT, 0, st>>>(in, out, ff, Ng, g, device_dt ? R(0) : dt / dh, gamma, order,
                                                   device_dt ? static_cast<const R*>(o->max_speed) : nullptr, device_dt ? (R)o->cfl : R(0),
                                                   static_cast<R*>(o->workspace), o->status);
  return (int)cudaGetLastError();
}

// ---- hydro_rtvd_solve_noalloc_f64: the scratch-slot kernel above with its scratch in a file-scope device array, for callers
// that cannot allocate (CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc).  Every GPU that loads the
// library holds the array (16.3 MiB) until exit.  The array's NAME is a host-side stand-in in host code, not a device address:
// the address comes from cudaGetSymbolAddress, once per device, with that device current.
constexpr int NOALLOC_SLOTS = 32;  // CTAs of the launch, one scratch slot each
constexpr size_t NOALLOC_SLOT_BYTES = 5 * ((size_t)RT_W * RT_W * PS + (size_t)RT_W * PS * PS) * sizeof(double);  // 535 040
static __device__ __align__(256) unsigned char g_rtvd_noalloc_scratch[NOALLOC_SLOTS * NOALLOC_SLOT_BYTES];
constexpr int NOALLOC_MAX_DEVICES = 64;

static int rtvd_noalloc_impl(const double* in, double* out, double* ff, int Ng, double dt, double dh, double gamma, int order,
                             long long* status, cudaStream_t st) {
  if (Ng < 0) return HYDRO_E_COUNT;
  if (Ng > HYDRO_RTVD_NOALLOC_MAX_GROUPS) return HYDRO_E_TOOBIG;
  if (order < 0 || order > 1) return HYDRO_E_ENUM;
  if (!(gamma > 1.0) || !(dh > 0.0) || !(dt >= 0.0)) return HYDRO_E_VALUE;
  if (Ng == 0) return HYDRO_OK;
  if (!in || !out) return HYDRO_E_NULL;
  if (((uintptr_t)in & 15) || ((uintptr_t)out & 15) || ((uintptr_t)ff & 15) || ((uintptr_t)status & 7)) return HYDRO_E_ALIGN;
  // set-up, once per device: the device address of the array on the CURRENT device (no allocation: the array is part of the
  // loaded module).  A benign race between two host threads writes the same value twice.
  static double* addr[NOALLOC_MAX_DEVICES] = {nullptr};
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return (int)e;
  if (dev < 0 || dev >= NOALLOC_MAX_DEVICES) return HYDRO_E_VALUE;
  double* scratch = addr[dev];
  if (!scratch) {
    void* ptr = nullptr;
    e = cudaGetSymbolAddress(&ptr, g_rtvd_noalloc_scratch);
    if (e != cudaSuccess) return (int)e;
    if (!ptr) return (int)cudaErrorInvalidSymbol;
    scratch = static_cast<double*>(ptr);
    addr[dev] = scratch;
  }
  // nothing in the scratch must start at zero: every sweep writes the whole range the next sweep reads, so the contents the
  // previous call left are never read
  const int slots = Ng < NOALLOC_SLOTS ? Ng : NOALLOC_SLOTS;
  rtvd_kernel<double, SPLIT_RTVD><<<(unsigned)slots, RT_NT, 0, st>>>(in, out, ff, Ng, RT_G, dt / dh, gamma, order, nullptr, 0.0, scratch, status);
  return (int)cudaGetLastError();
}

}  // namespace hydro

extern "C" {
int hydro_rtvd_solve_noalloc_f64(const double* in, double* out, double* face_flux, int Ng, double dt, double dh, double gamma, int order,
                                 long long* status, hydro_stream_t stream) {
  return hydro::rtvd_noalloc_impl(in, out, face_flux, Ng, dt, dh, gamma, order, status, (cudaStream_t)stream);
}
size_t hydro_rtvd_workspace_bytes(int Ng, int precision_bytes) {
  if (Ng <= 0 || (precision_bytes != 4 && precision_bytes != 8)) return 0;
  const size_t slots = Ng < hydro::RT_MAX_SLOTS ? (size_t)Ng : (size_t)hydro::RT_MAX_SLOTS;
  return slots * hydro::rtvd_slot_bytes((size_t)precision_bytes);
}
int hydro_rtvd_solve_f32(const float* in, float* out, float* face_flux, int Ng, float dt, float dh, float gamma, int order,
                         const hydro_opts* opts, hydro_stream_t stream) {
  return hydro::rtvd_impl<float>(in, out, face_flux, Ng, dt, dh, gamma, order, opts, (cudaStream_t)stream);
}
int hydro_rtvd_solve_f64(const double* in, double* out, double* face_flux, int Ng, double dt, double dh, double gamma, int order,
                         const hydro_opts* opts, hydro_stream_t stream) {
  return hydro::rtvd_impl<double>(in, out, face_flux, Ng, dt, dh, gamma, order, opts, (cudaStream_t)stream);
}
int hydro_waf_solve_f32(const float* in, float* out, float* face_flux, int Ng, float dt, float dh, float gamma, int order,
                        const hydro_opts* opts, hydro_stream_t stream) {
  return hydro::rtvd_impl<float>(in, out, face_flux, Ng, dt, dh, gamma, order, opts, (cudaStream_t)stream, hydro::SPLIT_WAF);
}
int hydro_waf_solve_f64(const double* in, double* out, double* face_flux, int Ng, double dt, double dh, double gamma, int order,
                        const hydro_opts* opts, hydro_stream_t stream) {
  return hydro::rtvd_impl<double>(in, out, face_flux, Ng, dt, dh, gamma, order, opts, (cudaStream_t)stream, hydro::SPLIT_WAF);
}
}
