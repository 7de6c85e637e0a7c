// hydro_lean_vl.cuh -- fused z-marching VL kernel (the half-step state comes from first-order
// Riemann fluxes of the cell-centred states, taken BEFORE the reconstruction; six Riemann solves per cell, S12).
//
// Two software-pipelined stages march along z through one persistent CTA per SM:
//   stage 1, plane a (the "plus" of cells within E = RW+1 of the interior along one axis):
//     S1  F1_x, F1_y at the lower faces of every plus cell (an extra warp solves the upper boundary faces),
//         F1_z(a) = RS(W(a-1), W(a)) column-local                                              | barrier 1
//     S2  U^{n+1/2}(a-1) = U - (nu/2)[dF1_x + dF1_y + (F1_z(a) - F1_z(a-1))] -> W-half ring     | barrier 2
//   stage 2, plane b = a - 1 - RW (the 18 x 18 tile minus corners, as in the MHM kernel):
//     S3  untraced face states of W-half in x, y, z -> LOX UPX LOY UPY; F_z(b) = RS(up_z(b-1), lo_z(b)),
//         boundary-flux store, conservative update and store of plane b-1                      | barrier 3
//     S4  F_x(b), F_y(b) -> FX, FY, boundary-flux stores; con->prim of raw plane a+1           | barrier 4
//     S5  carried D_z = (dF_x + dF_y)(b) - F_z(b)
// The first-pass flux fields alias LOX..UPY (disjoint lifetimes).  Plane feed and packed fields as in
// hydro_lean_ctu.cuh.
#pragma once
#include <cstdint>
#include "hydro_launch.cuh"
#include "hydro_lean_mhm.cuh"
#include "hydro_lean_grid.cuh"

namespace hydro {

template <class R, int RECON, int RS, int FAST, int GRID, int MERGE, int SPLIT>
__global__ void __launch_bounds__(VL_NT(RECON) + 320 * SPLIT, 1)
vl_lean_kernel(const R* __restrict__ in, R* __restrict__ out, R* __restrict__ face_flux, int Ng, int g_arg, Par<R> p,
               const R* __restrict__ max_speed, R cfl, long long* status, GridIO<R> gio) {
  using Op = LeanOps<R, RECON, RS, FAST>;
  using Mo = MhmOps<R, RECON, RS, FAST>;
  constexpr int RW = 1 + RECON, E = RW + 1, GW = E + 1, NW = 2 * RW + 1, NPL = PS + 2 * GW;
  constexpr int SW = PS + 2 * GW, WPL = SW * SW;        // primitive plane (stage 1 input)
  constexpr int SH = PS + 2 * E, HPL = SH * SH;         // W-half plane
  constexpr int SF = PS + 2 * E + 1, FPL = (SF * SF + 3) / 4 * 4;  // first-pass flux grid (one more face than cells per row)
  constexpr int NC = LEAN_COLS, FT = PS + 2;
  constexpr int NP = 320 + 64 * (E - 1);                // plus cells; then one warp of boundary-face jobs
  // SPLIT: the two stages run on warps of their own -- threads 0..319 the stage-2 columns, the next NP threads the stage-1 plus
  // cells, then the boundary warp: 23 (25) warps instead of 13 (15) hide each other's latencies (a thread has ONE role, so its
  // carried values share registers)
  constexpr int S1 = SPLIT ? 320 : 0;              // first stage-1 thread
  constexpr int NT = 320 + 64 * (RECON + 1) + 32 + S1;  // == VL_NT(RECON) + 320 SPLIT
  static_assert(2 * FPL <= 4 * NC, "first-pass flux fields must fit in LOX..UPY");
  // MERGE: the two stages share their barrier intervals (two CTA barriers per plane instead of four): stage 2 then runs one more
  // plane behind (b = a - 2 - RW) and the first-pass fluxes get their own fields.  The W-half ring needs no extra plane: S2
  // overwrites plane b - RW in the interval AFTER the one in which S3 read it for the last time.
  constexpr int NH = NW;
  apply_device_dt(p, max_speed, cfl);

  const int g = GRID ? GW : g_arg;  // grid mode: the ghost zones come from the grid, always at the minimum width
  const int S = PS + 2 * g;
  const int SS = S * S;
  const size_t nS = (size_t)SS * S;
  const int off = g - GW;
  const size_t N2 = (size_t)(gio.Gy * PS) * (gio.Gx * PS), N3 = N2 * (gio.Gz * PS);  // grid mode: plane / variable strides

  extern __shared__ __align__(16) unsigned char smem[];
  uint64_t* bar = reinterpret_cast<uint64_t*>(smem);   // [2]
  R* wpl = reinterpret_cast<R*>(smem + 64);            // one field of WPL cells: primitive plane a (W(a-1) lives in registers)
  R* hring = wpl + 5 * WPL;                       // [NH] fields of HPL cells: W-half planes b-RW .. b+RW
  R* xy = hring + NH * 5 * HPL;                        // [6] fields of NC cells: LOX UPX LOY UPY FX FY
  R* f1own = xy + 6 * 5 * NC;                          // MERGE: [2] fields of FPL cells, the first-pass fluxes
  R* raw = f1own + (MERGE ? 2 * 5 * FPL : 0);          // [5][SS] one landing plane: a step is long against a plane load
  R* f1x = MERGE ? f1own : xy;                         // not merged: the first-pass fluxes alias LOX.. (disjoint lifetimes)
  R* f1y = f1x + 5 * FPL;
  auto fld = [&](int k) { return xy + k * 5 * NC; };

  const int tid = threadIdx.x;
  // ---- stage-1 role: plus cell (ci, cj) in interior coordinates, or a boundary-face job of the extra warp
  int ci = 0, cj = 0;
  const int k1 = (SPLIT && tid >= S1) ? tid - S1 : tid;  // index within the stage's own numbering (the two coincide unless SPLIT)
  const bool cell = tid >= S1 && k1 < NP;
  if (k1 < PS * PS) { cj = k1 >> 4; ci = k1 & 15; }                                            // interior columns
  else if (k1 < PS * PS + 32) { const int l = k1 - PS * PS; cj = l >> 1; ci = (l & 1) ? PS : -1; }  // x ring
  else if (k1 < 320) { const int l = k1 - PS * FT; cj = (l < PS) ? -1 : PS; ci = l & (PS - 1); }    // y ring
  else if (cell) {
    const int k = k1 - 320, r = 2 + k / 64, arm = (k & 63) >> 4, pos = k & 15;
    ci = arm == 0 ? -r : (arm == 1 ? PS - 1 + r : pos);
    cj = arm == 2 ? -r : (arm == 3 ? PS - 1 + r : pos);
  }
  const bool c_int = cell && ci >= 0 && ci < PS && cj >= 0 && cj < PS;
  const bool bndw = tid >= S1 + NP;  // the boundary warp
  const int bl = tid - (S1 + NP);    // its lane
  // ---- stage-2 role (tid < 320): column of the 18 x 18 tile, as in the CTU / MHM kernels
  const int ii = ci + 1, jj = cj + 1;
  const bool s2 = tid < 320;
  const int col = jj * FT + ii;
  const bool in_i = s2 && ii >= 1 && ii <= PS, in_j = s2 && jj >= 1 && jj <= PS, interior = in_i && in_j;
  const int wb = (cj + GW) * SW + (ci + GW), hb = (cj + E) * SH + (ci + E), fb = (cj + E) * SF + (ci + E);

  const int my_groups = (Ng - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x;
  const int total_planes = my_groups * NPL;
  auto issue = [&](int n) {  // thread 0 only
    if (n >= total_planes) return;
    const int m = n / NPL, pl = n - m * NPL;
    const size_t grp = (size_t)blockIdx.x + (size_t)m * gridDim.x;
    const R* src = in + grp * 5 * nS + (size_t)(pl + off) * SS;
    uint64_t* b = bar;
    R* dst = raw;
    mbar_expect_tx(b, (uint32_t)(5 * SS * sizeof(R)));
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
  GridFeed<R, SW, NPL, NT> gf;
  gf.reset();
  if (GRID) gf.feed(gio, my_groups, raw, tid);
  else if (tid == 0) issue(0);

  Cnt c = {0, 0, 0};
  typename Bits<R>::U best = 0;  // running maximum of the updated cells' wave speed (next_max_speed)
  int nseq = 0;
  // grid mode: a thread waits for its own copies of the raw plane; the CTA barrier that follows publishes the plane
  auto landed = [&]() { if (GRID) cp_async_wait<0>(); };
  auto convert = [&]() {
    if (!GRID) mbar_wait(bar, (uint32_t)(nseq & 1));
    const R* rp = raw;
    R* wp = wpl;
    for (int idx = tid; idx < WPL; idx += NT) {
      const int b = idx / SW, a = idx - b * SW;
      stv(wp, WPL, idx, Op::c2p(ld5(rp + (b + off) * S + (a + off), SS), p, c));
    }
  };
  auto refill = [&]() {
    if (GRID) gf.feed(gio, my_groups, raw, tid);
    else if (tid == 0) { fence_async_smem(); issue(nseq + 1); }
    ++nseq;
  };

  V5<R> Wprev, s1prev, f1zprev, uzc_own, Dz_own;  // W(a-1); (dF1_x + dF1_y)(a-1); F1_z(a-1); up_z(b-1); (dF_x + dF_y - F_z)(b-1)
#pragma unroll
  for (int q = 0; q < 5; ++q) { Wprev[q] = R(1); s1prev[q] = R(0); f1zprev[q] = R(0); uzc_own[q] = R(0); Dz_own[q] = R(0); }
  // SPLIT: a thread carries either the stage-1 or the stage-2 values: the latter live in the former's registers
  V5<R>& uzc = SPLIT ? Wprev : uzc_own;
  V5<R>& Dz = SPLIT ? s1prev : Dz_own;

  for (int m = 0; m < my_groups; ++m) {
    const size_t grp = (size_t)blockIdx.x + (size_t)m * gridDim.x;
    const R* gin0 = in + grp * 5 * nS + ((size_t)g * S + (cj + g)) * S + (ci + g);
    R* gout0 = out + grp * 5 * PS * PS * PS + cj * PS + ci;
    if (GRID) {  // U^n and the result live in the grids (interior columns only)
      const size_t cell0 = (c_int || interior) ? grid_cell0(gio, grp, ci, cj) : 0;
      gin0 = gio.gin + cell0;
      gout0 = gio.gout + cell0;
    }
    const size_t pstr_in = GRID ? N2 : (size_t)SS, vstr_in = GRID ? N3 : nS;
    R* gff = face_flux ? face_flux + grp * 9 * 5 * PS * PS : nullptr;
    // ---- prologue: plane -GW (only its own-column values are needed, as W(a-1) of the first step), then plane -E
    if (GRID) { landed(); __syncthreads(); }
    convert();
    __syncthreads();
    refill();
    if (c_int) Wprev = ldv(wpl, WPL, wb);
    if (GRID) landed();
    __syncthreads();
    convert();
    __syncthreads();
    refill();

#pragma unroll 1
    for (int a = -E; a <= PS + E + MERGE; ++a) {
      const bool a_s1 = !MERGE || a <= PS + E;     // merged: one more step, which only drains stage 2
      const bool a_in = a >= 0 && a < PS;          // plane a holds arm cells
      const bool a_xy = a < PS + E;                // plane a needs its in-plane first-pass fluxes
      const R* wa = wpl;
      // arm cells (outside the interior columns) live in planes 0..15 only, but need W(-1) and F1_z at faces 0 and 16
      const bool act1 = a_s1 && cell && (c_int || (a >= -1 && a <= PS));
      const bool zf = a_s1 && cell && (c_int || (a >= 0 && a <= PS));
      const bool xyf = cell && a_xy && (c_int || a_in);
      const int b = a - 1 - RW - MERGE;            // plane of stage 2
      const bool b_in = b >= 0 && b < PS;
      const bool conv = a + 1 <= PS - 1 + GW;      // plane a+1 replaces plane a in S4 (last read in S1)
      V5<R> W0, f1z;
      auto stage1 = [&]() {
      // ================= S1: first-order fluxes of plane a =================
      if (act1) {
        W0 = ldv(wa, WPL, wb);
        if (xyf) {
          stv(f1x, FPL, fb, Op::template riemann<0>(ldv(wa, WPL, wb - 1), W0, p, c));
          stv(f1y, FPL, fb, Op::template riemann<1>(ldv(wa, WPL, wb - SW), W0, p, c));
        }
        if (zf) f1z = Op::template riemann<2>(Wprev, W0, p, c);
      } else if (bndw && a_xy) {
        // boundary warp: the upper faces that no plus cell owns.  Inner plane: x (16+E, l) / y (l, 16+E) for l < 16 and the
        // 2E arm-only rows / columns r: x (16, r) / y (r, 16).  Outer plane (interior columns only): x (16, l) / y (l, 16).
        int r = -100, edge = PS;
        if (bl < PS) { r = bl; edge = a_in ? PS + E : PS; }
        else if (a_in && bl < PS + 2 * E) { const int k = bl - PS; r = k < E ? k - E : PS + (k - E); }
        if (r != -100) {
          const int xw = (r + GW) * SW + (edge + GW), yw = (edge + GW) * SW + (r + GW);
          stv(f1x, FPL, (r + E) * SF + (edge + E), Op::template riemann<0>(ldv(wa, WPL, xw - 1), ldv(wa, WPL, xw), p, c));
          stv(f1y, FPL, (edge + E) * SF + (r + E), Op::template riemann<1>(ldv(wa, WPL, yw - SW), ldv(wa, WPL, yw), p, c));
        }
      }
      };
      auto stage2 = [&]() {
      // ================= S2: half-step state of plane a-1 -> W-half ring =================
      if (act1) {
        V5<R> s1;
#pragma unroll
        for (int q = 0; q < 5; ++q) s1[q] = R(0);
        if (xyf) {
          const V5<R> x1 = ldv(f1x, FPL, fb + 1), x0 = ldv(f1x, FPL, fb), y1 = ldv(f1y, FPL, fb + SF), y0 = ldv(f1y, FPL, fb);
#pragma unroll
          for (int q = 0; q < 5; ++q) s1[q] = (x1[q] - x0[q]) + (y1[q] - y0[q]);
        }
        const int ap = a - 1;  // plane whose half step is complete now
        const bool ap_in = ap >= 0 && ap < PS;
        if (ap >= -E && (ap_in || c_int)) {
          // U^n of plane a-1 (the half step starts from U^n): rebuilt from the primitives held in registers, which
          // is U^n to rounding -- unless a floor changed them: then the raw conserved state is re-read (L2-resident)
          V5<R> U;
          if (!FAST && (p.min_dens > R(0) || p.min_pres > R(0))) {
            // (the arm cells of a floored grid-mode run would need folded addresses: hydro_solve_grid_* does not take floors with VL)
            const R* gp = gin0 + (ptrdiff_t)ap * (ptrdiff_t)pstr_in;
#pragma unroll
            for (int q = 0; q < 5; ++q) { U[q] = __ldg(gp); gp += vstr_in; }
          } else {
            U = prim2cons(Wprev, p);
          }
#pragma unroll
          for (int q = 0; q < 5; ++q) U[q] = U[q] - p.hnu * (s1prev[q] + (f1z[q] - f1zprev[q]));
          stv(hring + ((ap + E) % NH) * 5 * HPL, HPL, hb, Op::c2p(U, p, c));
        }
        Wprev = W0;
        s1prev = s1;
        f1zprev = f1z;
      }
      };
      auto stage3 = [&]() {
      // ================= S3: face states of W-half plane b, F_z(b), update of plane b-1 =================
      if (s2 && b >= -1 && (b_in || interior)) {
        V5<R> Uold;
        const bool upd = interior && b >= 1;
        if (upd) {
          const R* gin = gin0 + (size_t)(b - 1) * pstr_in;
#pragma unroll
          for (int q = 0; q < 5; ++q) { Uold[q] = __ldg(gin); gin += vstr_in; }
        }
        const R* hp = hring + ((b + E) % NH) * 5 * HPL;
        const V5<R> H0 = ldv(hp, HPL, hb);
        if (b_in && in_j) {
          const V5<R> Wb = ldv(hp, HPL, hb - 1), Wc = ldv(hp, HPL, hb + 1);
          V5<R> Wa = Wb, Wd = Wc, l, u;
          if (RECON == RECON_PPM) { Wa = ldv(hp, HPL, hb - 2); Wd = ldv(hp, HPL, hb + 2); }
          Mo::template recon<0>(Wa, Wb, H0, Wc, Wd, p, l, u);
          stv(fld(LF_LOX), NC, col, l);
          stv(fld(LF_UPX), NC, col, u);
        }
        if (b_in && in_i) {
          const V5<R> Wb = ldv(hp, HPL, hb - SH), Wc = ldv(hp, HPL, hb + SH);
          V5<R> Wa = Wb, Wd = Wc, l, u;
          if (RECON == RECON_PPM) { Wa = ldv(hp, HPL, hb - 2 * SH); Wd = ldv(hp, HPL, hb + 2 * SH); }
          Mo::template recon<1>(Wa, Wb, H0, Wc, Wd, p, l, u);
          stv(fld(LF_LOY), NC, col, l);
          stv(fld(LF_UPY), NC, col, u);
        }
        if (interior) {
          const V5<R> Wb = ldv(hring + ((b - 1 + E) % NH) * 5 * HPL, HPL, hb), Wc = ldv(hring + ((b + 1 + E) % NH) * 5 * HPL, HPL, hb);
          V5<R> Wa = Wb, Wd = Wc, lz, uz;
          if (RECON == RECON_PPM) {
            Wa = ldv(hring + ((b - 2 + E) % NH) * 5 * HPL, HPL, hb);
            Wd = ldv(hring + ((b + 2 + E) % NH) * 5 * HPL, HPL, hb);
          }
          Mo::template recon<2>(Wa, Wb, H0, Wc, Wd, p, lz, uz);
          if (b >= 0) {
            const V5<R> Fz = Op::template riemann<2>(uzc, lz, p, c);
            if (gff && (b & 7) == 0) st5(gff + (size_t)((6 + (b >> 3)) * 5) * 256 + cj * PS + ci, 256, Fz);
            if (upd) {
              V5<R> U;
#pragma unroll
              for (int q = 0; q < 5; ++q) U[q] = Uold[q] - p.nu * (Dz[q] + Fz[q]);
              const V5<R> Wn = Op::c2p(U, p, c);
              if (p.next_speed) track_speed(Wn, p, best);
              if (!FAST && (p.min_dens > R(0) || p.min_pres > R(0))) U = prim2cons(Wn, p);
              if (GRID) {
                R* d = gout0 + (size_t)(b - 1) * N2;
#pragma unroll
                for (int q = 0; q < 5; ++q) { *d = U[q]; d += N3; }
              } else {
                st5(gout0 + (b - 1) * PS * PS, PS * PS * PS, U);
              }
            }
            Dz = Fz;
          }
          if (b < PS) uzc = uz;
        }
      }
      };
      auto stage4 = [&]() {
      // ================= S4: F_x(b), F_y(b), boundary-flux stores; con->prim of plane a+1 =================
      if (s2 && b_in) {
        if (in_j && ii >= 1) {
          const V5<R> f = Op::template riemann<0>(ldv(fld(LF_UPX), NC, col - 1), ldv(fld(LF_LOX), NC, col), p, c);
          stv(fld(LF_FX), NC, col, f);
          if (gff && ((ii - 1) & 7) == 0) st5(gff + (size_t)(((ii - 1) >> 3) * 5) * 256 + b * PS + (jj - 1), 256, f);
        }
        if (in_i && jj >= 1) {
          const V5<R> f = Op::template riemann<1>(ldv(fld(LF_UPY), NC, col - FT), ldv(fld(LF_LOY), NC, col), p, c);
          stv(fld(LF_FY), NC, col, f);
          if (gff && ((jj - 1) & 7) == 0) st5(gff + (size_t)((3 + ((jj - 1) >> 3)) * 5) * 256 + b * PS + (ii - 1), 256, f);
        }
      }
      };
      auto stage5 = [&](bool bin5) {
      // ================= S5: carried x+y flux difference of plane b minus F_z(b) =================
      if (bin5 && interior) {
        const V5<R> x1 = ldv(fld(LF_FX), NC, col + 1), x0 = ldv(fld(LF_FX), NC, col);
        const V5<R> y1 = ldv(fld(LF_FY), NC, col + FT), y0 = ldv(fld(LF_FY), NC, col);
#pragma unroll
        for (int q = 0; q < 5; ++q) Dz[q] = ((x1[q] - x0[q]) + (y1[q] - y0[q])) - Dz[q];
      }
      };
      if (MERGE) {
        // two barrier intervals per plane: {S5 of the previous plane, S1 of plane a, S3 of plane b} | {S2, S4, con->prim}
        stage5(b - 1 >= 0 && b - 1 < PS);
        stage1();
        stage3();
        if (conv) landed();
        __syncthreads();  // barrier 1
        stage2();
        stage4();
        if (conv) convert();
        __syncthreads();  // barrier 2
        if (conv) refill();
      } else {
        stage1();
        __syncthreads();  // barrier 1
        stage2();
        __syncthreads();  // barrier 2
        stage3();
        if (conv) landed();
        __syncthreads();  // barrier 3
        stage4();
        if (conv) convert();  // plane a+1 replaces plane a, read for the last time in S1
        __syncthreads();  // barrier 4
        if (conv) refill();
        stage5(b_in);
      }
    }
  }
  flush_counters(c, status);
  flush_speed(best, p.next_speed);
}

template <class R, int RECON, int RS, int FAST, int GRID = 0> cudaError_t launch_vl_lean(const SolveArgs<R>& a) {
  constexpr int SPLIT = vl_split(sizeof(R), RECON, RS) ? 1 : 0;
  auto kern = vl_lean_kernel<R, RECON, RS, FAST, GRID, vl_merged(sizeof(R), RECON) ? 1 : 0, SPLIT>;
  const size_t smem = vl_smem_bytes(sizeof(R), RECON, a.g);
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
  kern<<<(unsigned)grid, VL_NT(RECON) + 320 * SPLIT, smem, a.stream>>>(a.in, a.out, a.face_flux, a.Ng, a.g, a.par, a.max_speed, a.cfl, a.status, a.grid);
  return cudaGetLastError();
}

}  // namespace hydro
