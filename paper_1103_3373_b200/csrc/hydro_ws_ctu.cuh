// hydro_ws_ctu.cuh -- warp-specialised fused CTU kernel (steps (1)-(5) in one launch).
//
// Same z-marching organisation as hydro_fused_ctu.cuh (one persistent CTA per SM, planes streamed by
// 1-D bulk async copies, every intermediate on chip), but the work of a plane is split between two
// warp groups that run concurrently and meet only at a double-buffered hand-off in shared memory:
//
//   group P ("predictor", 11 warps): steps (1)-(2) of PAPER.md:39-40 and the flux differences of (3).
//       One thread per column of the 18 x 18 tile (interior + one-cell ring).  Per plane t:
//       con->prim of plane t+LA into the primitive ring; traced z states of plane t+1 and F*_z(t+1)
//       (column-local, carried in registers); traced x,y states of plane t; F*_x(t), F*_y(t); then the
//       three half-step transverse increments of the cell (S4: half nu, cyclic t1,t2)
//           dq_x = (nu/2)(dF*_y + dF*_z),  dq_y = (nu/2)(dF*_z + dF*_x),  dq_z = (nu/2)(dF*_x + dF*_y).
//       The six traced face states and the three increments (45 values per column) are the hand-off.
//   group C ("corrector", 9 warps): steps (3)-(5).  One thread per FACE: it corrects the
//       two states that meet at its face (U <- U - dq of the state's own cell), solves the second
//       Riemann problem, stores patch-boundary fluxes, and (z-face threads, which own a column) forms
//       the conservative update of the plane below.  Faces are compacted onto threads: 256 z + 272 x +
//       272 y faces per plane on 288 threads.
//
// Why: the single-role kernel carries ~70 values per thread from stage to stage and ends at 168
// registers x 352 threads = 11 warps per SM, issue slots half empty (profiles/r1_ncu_fused_f32_v1.md).
// Splitting the plane at the hand-off leaves each role ~25 carried values, so 20 warps fit at 96
// registers, the two roles overlap each other's barriers, and pass-2 lanes are no longer idle on the
// ring columns.  The arithmetic is the same device code (hydro_math.cuh) in the same order.
//
// Synchronisation: named barriers (bar.sync 1 / 2) inside each group; mbarriers full[2] / empty[2]
// (acquire/release at CTA scope) for the hand-off; mbarriers tma[2] for the plane loads.
#pragma once
#include <cstdint>
#include "hydro_fused_ctu.cuh"

namespace hydro {

// transverse correction of one face state: W <- prim(cons(W) - dq)
template <class R> __device__ __forceinline__ V5<R> ctu_correct(const V5<R>& W, const V5<R>& dq, const Par<R>& p, Cnt& c) {
  V5<R> U = prim2cons(W, p);
#pragma unroll
  for (int q = 0; q < 5; ++q) U[q] = U[q] - dq[q];
  return cons2prim(U, p, c);
}

// hand-off record kinds (each [5][WS_COLS])
enum : int { HK_LOX = 0, HK_UPX, HK_LOY, HK_UPY, HK_LOZ, HK_UPZ, HK_DQX, HK_DQY, HK_DQZ, HK_N };

template <class R, int RECON, int RS>
__global__ void __launch_bounds__(WS_NT, 1)
ctu_ws_kernel(const R* __restrict__ in, R* __restrict__ out, R* __restrict__ face_flux, int Ng, int g, Par<R> p,
              const R* __restrict__ max_speed, R cfl, long long* status) {
  constexpr int GW = 2 + RECON, RW = 1 + RECON, LA = RW + 1, SWP = PS + 2 * GW, NW = 2 * RW + 1, NPL = PS + 2 * GW;
  constexpr int WPL = SWP * SWP;
  constexpr int NC = WS_COLS;      // 324 columns, c = jj * 18 + ii
  constexpr int NHP = PS + 2;      // planes handed off per group: t = -1 .. 16
  apply_device_dt(p, max_speed, cfl);

  const int S = PS + 2 * g;
  const int SS = S * S;
  const size_t nS = (size_t)SS * S;
  const int off = g - GW;

  extern __shared__ __align__(16) unsigned char smem[];
  uint64_t* bar_tma = reinterpret_cast<uint64_t*>(smem);  // [2]
  uint64_t* bar_full = bar_tma + 2;                       // [2]
  uint64_t* bar_empty = bar_tma + 4;                      // [2]
  R* raw = reinterpret_cast<R*>(smem + 64);               // [2][5][SS]
  R* ring = raw + (size_t)2 * 5 * SS;                     // [NW][5][WPL]
  R* hand = ring + (size_t)NW * 5 * WPL;                  // [2][HK_N][5][NC]
  R* xch = hand + (size_t)2 * HK_N * 5 * NC;              // [2][5][NC]      F*_x, F*_y (group P)
  R* fbuf = xch + (size_t)2 * 5 * NC;                     // [2][2][5][NC]   F_x, F_y (group C), double-buffered

  const int tid = threadIdx.x;
  if (tid == 0) {
    mbar_init(bar_tma, 1);
    mbar_init(bar_tma + 1, 1);
    mbar_init(bar_full, WS_NT1);
    mbar_init(bar_full + 1, WS_NT1);
    mbar_init(bar_empty, WS_NT2);
    mbar_init(bar_empty + 1, WS_NT2);
    fence_mbar_init();
    fence_async_smem();
  }
  __syncthreads();

  const int my_groups = (Ng - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x;
  Cnt c = {0, 0, 0};

  if (tid < WS_NT1) {
    // =========================== group P: reconstruction, first Riemann pass, dq ===========================
    int ii, jj;
    bool valid = tid < NC, corner = false;
    if (tid < PS) { ii = tid + 1; jj = 0; }
    else if (tid < PS + PS * FT) { const int r = tid - PS; jj = 1 + r / FT; ii = r % FT; }
    else if (tid < 2 * PS + PS * FT) { ii = tid - (PS + PS * FT) + 1; jj = FT - 1; }
    else { corner = true; ii = (tid & 1) ? FT - 1 : 0; jj = (tid & 2) ? FT - 1 : 0; }
    const int col = jj * FT + ii;
    const bool regular = valid && !corner;
    const bool in_i = valid && ii >= 1 && ii <= PS, in_j = valid && jj >= 1 && jj <= PS;
    const bool interior = in_i && in_j;
    const int wb = (jj + GW - 1) * SWP + (ii + GW - 1);

    const int total_planes = my_groups * NPL;
    const uint32_t plane_bytes = (uint32_t)(5 * SS * sizeof(R));
    auto issue = [&](int n) {  // thread 0 only
      if (n >= total_planes) return;
      const int m = n / NPL, pl = n % NPL;
      const size_t grp = (size_t)blockIdx.x + (size_t)m * gridDim.x;
      const R* src = in + grp * 5 * nS + (size_t)(pl + off) * SS;
      uint64_t* b = bar_tma + (n & 1);
      R* dst = raw + (size_t)(n & 1) * 5 * SS;
      mbar_expect_tx(b, plane_bytes);
#pragma unroll
      for (int q = 0; q < 5; ++q) bulk_g2s(dst + (size_t)q * SS, src + q * nS, (uint32_t)(SS * sizeof(R)), b);
    };
    if (tid == 0) { issue(0); issue(1); }

    V5<R> zlo_c, zup_c, f1z_c;  // traced z states of plane t and F*_z at its lower face (carried along the column)
    int nseq = 0, hseq = 0;
    for (int m = 0; m < my_groups; ++m) {
      for (int t = -GW - LA; t <= PS; ++t) {
        // ---- A: con->prim of plane t+LA into the ring
        const int pc = t + LA;
        if (pc <= PS - 1 + GW) {
          const int st = nseq & 1;
          mbar_wait(bar_tma + st, (uint32_t)((nseq >> 1) & 1));
          const R* rp = raw + (size_t)st * 5 * SS;
          R* wp = ring + (size_t)((pc + GW) % NW) * 5 * WPL;
          for (int idx = tid; idx < WPL; idx += WS_NT1) {
            const int a = idx % SWP, b = idx / SWP;
            const V5<R> U = ld5(rp + (b + off) * S + (a + off), SS);
            st5(wp + idx, WPL, cons2prim(U, p, c));
          }
        }
        group_bar<1, WS_NT1>();
        if (pc <= PS - 1 + GW) {
          if (tid == 0) { fence_async_smem(); issue(nseq + 2); }
          ++nseq;
        }
        if (t < -2) continue;

        // ---- B: traced z states of plane t+1, F*_z(t+1) = RS(up_z(t), lo_z(t+1))
        const int kz = t + 1;
        V5<R> lz, uz, f1z_n;
        if (regular && kz <= PS) {
          V5<R> Wz[2 * RW + 1];
#pragma unroll
          for (int s = 0; s < 2 * RW + 1; ++s)
            Wz[s] = to_normal<2>(ld5(ring + (size_t)((kz - RW + s + GW) % NW) * 5 * WPL + wb, WPL));
          V5<R> l, u;
          reconstruct<RECON, true>(Wz[0], Wz[RW - 1], Wz[RW], Wz[RW + 1], Wz[2 * RW], p, l, u);
          lz = from_normal<2>(l);
          uz = from_normal<2>(u);
          if (kz >= 0) f1z_n = riemann_d<RS, 2>(zup_c, lz, p, c);
        }
        if (t < -1) {
          zlo_c = lz; zup_c = uz; f1z_c = f1z_n;
          continue;
        }

        // ---- hand-off slot of plane t
        const int hb = hseq & 1;
        mbar_wait(bar_empty + hb, (uint32_t)(((hseq >> 1) & 1) ^ 1));
        R* H = hand + (size_t)hb * HK_N * 5 * NC + col;

        // ---- C: traced x,y states of plane t; z states of plane t
        if (valid) {
          const R* wt = ring + (size_t)((t + GW) % NW) * 5 * WPL + wb;
          const V5<R> W0 = ld5(wt, WPL);
          {
            const V5<R> Wb = ld5(wt - 1, WPL), Wc = ld5(wt + 1, WPL);
            V5<R> Wa = Wb, Wd = Wc;
            if (RECON == RECON_PPM) { Wa = ld5(wt - 2, WPL); Wd = ld5(wt + 2, WPL); }
            V5<R> l, u;
            reconstruct<RECON, true>(to_normal<0>(Wa), to_normal<0>(Wb), to_normal<0>(W0), to_normal<0>(Wc), to_normal<0>(Wd), p, l, u);
            st5(H + HK_LOX * 5 * NC, NC, from_normal<0>(l));
            st5(H + HK_UPX * 5 * NC, NC, from_normal<0>(u));
          }
          {
            const V5<R> Wb = ld5(wt - SWP, WPL), Wc = ld5(wt + SWP, WPL);
            V5<R> Wa = Wb, Wd = Wc;
            if (RECON == RECON_PPM) { Wa = ld5(wt - 2 * SWP, WPL); Wd = ld5(wt + 2 * SWP, WPL); }
            V5<R> l, u;
            reconstruct<RECON, true>(to_normal<1>(Wa), to_normal<1>(Wb), to_normal<1>(W0), to_normal<1>(Wc), to_normal<1>(Wd), p, l, u);
            st5(H + HK_LOY * 5 * NC, NC, from_normal<1>(l));
            st5(H + HK_UPY * 5 * NC, NC, from_normal<1>(u));
          }
          if (interior) {
            st5(H + HK_LOZ * 5 * NC, NC, zlo_c);
            st5(H + HK_UPZ * 5 * NC, NC, zup_c);
          }
        }
        group_bar<1, WS_NT1>();

        // ---- D: F*_x(t), F*_y(t)
        V5<R> f1x, f1y;
        if (valid && ii >= 1) {
          f1x = riemann_d<RS, 0>(ld5(H + HK_UPX * 5 * NC - 1, NC), ld5(H + HK_LOX * 5 * NC, NC), p, c);
          st5(xch + col, NC, f1x);
        }
        if (valid && jj >= 1) {
          f1y = riemann_d<RS, 1>(ld5(H + HK_UPY * 5 * NC - FT, NC), ld5(H + HK_LOY * 5 * NC, NC), p, c);
          st5(xch + 5 * NC + col, NC, f1y);
        }
        group_bar<1, WS_NT1>();

        // ---- E: half-step transverse increments (S4)
        {
          const bool plane_in = (t >= 0 && t < PS);
          V5<R> dFx, dFy, dFz;
          if (in_i) {
            const V5<R> a = ld5(xch + col + 1, NC);
#pragma unroll
            for (int q = 0; q < 5; ++q) dFx[q] = a[q] - f1x[q];
          }
          if (in_j) {
            const V5<R> a = ld5(xch + 5 * NC + col + FT, NC);
#pragma unroll
            for (int q = 0; q < 5; ++q) dFy[q] = a[q] - f1y[q];
          }
          if (plane_in && regular) {
#pragma unroll
            for (int q = 0; q < 5; ++q) dFz[q] = f1z_n[q] - f1z_c[q];
          }
          if (in_j && plane_in) {
            V5<R> dq;
#pragma unroll
            for (int q = 0; q < 5; ++q) dq[q] = p.hnu * (dFy[q] + dFz[q]);
            st5(H + HK_DQX * 5 * NC, NC, dq);
          }
          if (in_i && plane_in) {
            V5<R> dq;
#pragma unroll
            for (int q = 0; q < 5; ++q) dq[q] = p.hnu * (dFz[q] + dFx[q]);
            st5(H + HK_DQY * 5 * NC, NC, dq);
          }
          if (interior) {
            V5<R> dq;
#pragma unroll
            for (int q = 0; q < 5; ++q) dq[q] = p.hnu * (dFx[q] + dFy[q]);
            st5(H + HK_DQZ * 5 * NC, NC, dq);
          }
        }
        mbar_arrive(bar_full + hb);
        ++hseq;
        zlo_c = lz; zup_c = uz; f1z_c = f1z_n;
      }
    }
  } else {
    // =========================== group C: correction, second Riemann pass, update ===========================
    const int ct = tid - WS_NT1;
    const bool zt = ct < PS * PS;                  // z faces / columns: (i, j)
    const int zi = ct & 15, zj = ct >> 4, zc = (zj + 1) * FT + zi + 1;
    const bool xt = ct < (PS + 1) * PS;            // x faces: f = 0..16 fastest, j
    const int xf = ct % (PS + 1), xj = ct / (PS + 1), xcr = (xj + 1) * FT + xf + 1;
    const bool yt = xt;                            // y faces: i fastest, f = 0..16
    const int yi = ct & 15, yf = ct >> 4, ycr = (yf + 1) * FT + yi + 1;

    V5<R> uzc, f2z, sxy, Uold;  // corrected up_z of the plane below; F_z at its lower face; its x+y flux difference; U^n
    int hseq = 0;
    for (int m = 0; m < my_groups; ++m) {
      const size_t grp = (size_t)blockIdx.x + (size_t)m * gridDim.x;
      const R* gin = in + grp * 5 * nS;
      R* gout = out + grp * 5 * PS * PS * PS;
      R* gff = face_flux ? face_flux + grp * 9 * 5 * PS * PS : nullptr;
      for (int t = -1; t <= PS; ++t) {
        const int hb = hseq & 1;
        mbar_wait(bar_full + hb, (uint32_t)((hseq >> 1) & 1));
        const R* H = hand + (size_t)hb * HK_N * 5 * NC;
        const bool plane_in = (t >= 0 && t < PS);
        R* Fx = fbuf + (size_t)((t & 1) * 2) * 5 * NC;
        R* Fy = Fx + 5 * NC;

        if (zt) {  // F_z(t) = RS(up_z'(t-1), lo_z'(t)); update of plane t-1
          const V5<R> dq = ld5(H + HK_DQZ * 5 * NC + zc, NC);
          if (t >= 0) {
            const V5<R> wl = ctu_correct(ld5(H + HK_LOZ * 5 * NC + zc, NC), dq, p, c);
            const V5<R> f2z_new = riemann_d<RS, 2>(uzc, wl, p, c);
            if (gff && (t & 7) == 0) st5(gff + (size_t)((6 + (t >> 3)) * 5) * 256 + ct, 256, f2z_new);
            if (t >= 1) {
              V5<R> U;
#pragma unroll
              for (int q = 0; q < 5; ++q) U[q] = Uold[q] - p.nu * (sxy[q] + (f2z_new[q] - f2z[q]));
              const V5<R> Wn = cons2prim(U, p, c);
              if (p.min_dens > R(0) || p.min_pres > R(0)) U = prim2cons(Wn, p);
              st5(gout + (t - 1) * PS * PS + ct, PS * PS * PS, U);
            }
            f2z = f2z_new;
          }
          if (t < PS) uzc = ctu_correct(ld5(H + HK_UPZ * 5 * NC + zc, NC), dq, p, c);
        }
        if (plane_in && xt) {  // F_x(t) at face xf of row xj
          const V5<R> wl = ctu_correct(ld5(H + HK_UPX * 5 * NC + xcr - 1, NC), ld5(H + HK_DQX * 5 * NC + xcr - 1, NC), p, c);
          const V5<R> wr = ctu_correct(ld5(H + HK_LOX * 5 * NC + xcr, NC), ld5(H + HK_DQX * 5 * NC + xcr, NC), p, c);
          const V5<R> f = riemann_d<RS, 0>(wl, wr, p, c);
          st5(Fx + xcr, NC, f);
          if (gff && (xf & 7) == 0) st5(gff + (size_t)((xf >> 3) * 5) * 256 + t * PS + xj, 256, f);
        }
        if (plane_in && yt) {  // F_y(t) at face yf of column yi
          const V5<R> wl = ctu_correct(ld5(H + HK_UPY * 5 * NC + ycr - FT, NC), ld5(H + HK_DQY * 5 * NC + ycr - FT, NC), p, c);
          const V5<R> wr = ctu_correct(ld5(H + HK_LOY * 5 * NC + ycr, NC), ld5(H + HK_DQY * 5 * NC + ycr, NC), p, c);
          const V5<R> f = riemann_d<RS, 1>(wl, wr, p, c);
          st5(Fy + ycr, NC, f);
          if (gff && (yf & 7) == 0) st5(gff + (size_t)((3 + (yf >> 3)) * 5) * 256 + t * PS + yi, 256, f);
        }
        mbar_arrive(bar_empty + hb);
        ++hseq;
        group_bar<2, WS_NT2>();
        if (zt && plane_in) {  // x+y flux difference of plane t; U^n of plane t for the update at t+1
#pragma unroll
          for (int q = 0; q < 5; ++q)
            sxy[q] = (Fx[q * NC + zc + 1] - Fx[q * NC + zc]) + (Fy[q * NC + zc + FT] - Fy[q * NC + zc]);
          const int xin = ((t + g) * S + (zj + g)) * S + (zi + g);
#pragma unroll
          for (int q = 0; q < 5; ++q) Uold[q] = __ldg(gin + q * nS + xin);
        }
      }
    }
  }
  flush_counters(c, status);
}

template <class R, int RECON, int RS> cudaError_t launch_ctu_ws(const SolveArgs<R>& a) {
  auto kern = ctu_ws_kernel<R, RECON, RS>;
  const size_t smem = ws_smem_bytes(sizeof(R), RECON, a.g);
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
  const int grid = a.Ng < sms ? a.Ng : sms;
  kern<<<(unsigned)grid, WS_NT, smem, a.stream>>>(a.in, a.out, a.face_flux, a.Ng, a.g, a.par, a.max_speed, a.cfl, a.status);
  return cudaGetLastError();
}

}  // namespace hydro
