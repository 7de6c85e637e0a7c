// hydro_lean_mhm.cuh -- fused z-marching MHM (MUSCL-Hancock) kernel: PAPER.md:35, 46, 93 -- steps (1)-(5) of
// PAPER.md:39-44 with the half-step of the face values taken from cell-local flux differences of all three
// directions, no Riemann solver in the predictor, three Riemann solves per cell.
//
// Same organisation as hydro_lean_ctu.cuh: persistent 320-thread CTAs (two per SM where the tiles allow),
// one thread per column of the 18 x 18 tile (MHM never touches the four corner columns), primitive planes in
// a ring fed by 1-D bulk async copies, packed "4+1" shared-memory fields.  MHM needs only two barriers per plane:
//   P1  untraced face states of plane t in x, y, z (S6/S7); Hancock increment (hnu * sum_d [F_d(W+_d) - F_d(W-_d)],
//       S13: one increment for the six face values of the cell); advanced x,y states -> LOX UPX LOY UPY;
//       z is column-local: F_z(t) = RS(up_z(t-1), lo_z(t)), boundary-flux store, conservative update and
//       store of plane t-1 as U - nu (D_z + F_z(t))                                               | barrier A
//   P2  F_x(t), F_y(t) -> FX, FY; patch-boundary flux stores; con->prim of the next raw plane     | barrier B
//   P3  carried D_z = (dF_x + dF_y)(t) - F_z(t)
#pragma once
#include <cstdint>
#include "hydro_launch.cuh"
#include "hydro_lean_ctu.cuh"
#include "hydro_lean_grid.cuh"

namespace hydro {

// untraced PLM face values, van Leer limiter on primitive variables (normal frame irrelevant: per component)
template <class R> __device__ __forceinline__ void lean_plm(const V5<R>& Wm, const V5<R>& W0, const V5<R>& Wp, V5<R>& lo, V5<R>& up) {
#pragma unroll
  for (int q = 0; q < 5; ++q) {
    const R h = vl_half_slope(W0[q] - Wm[q], Wp[q] - W0[q]);
    lo[q] = W0[q] - h;
    up[q] = W0[q] + h;
  }
}
// physical flux along D of an xyz-frame primitive state; (E + P) = gamma/(gamma-1) P + rho |v|^2 / 2
template <int D, class R> __device__ __forceinline__ V5<R> lean_phys_flux(const V5<R>& W, const Par<R>& p) {
  const R u = W[1 + D], m = W[0] * u;
  const R hq = R(0.5) * m_fma(W[3], W[3], m_fma(W[2], W[2], W[1] * W[1]));
  V5<R> F;
  F[0] = m;
  F[1] = m * W[1];
  F[2] = m * W[2];
  F[3] = m * W[3];
  F[1 + D] += W[4];
  F[4] = m_fma(m, hq, u * ((p.gamma * p.igm1) * W[4]));
  return F;
}

template <class R, int RECON, int RS, int FAST> struct MhmOps {
  using Op = LeanOps<R, RECON, RS, FAST>;
  // untraced face states of the middle cell along D (xyz-frame in and out)
  template <int D>
  static __device__ __forceinline__ void recon(const V5<R>& Wm2, const V5<R>& Wm1, const V5<R>& W0, const V5<R>& Wp1,
                                               const V5<R>& Wp2, const Par<R>& p, V5<R>& lo, V5<R>& up) {
    if (FAST && RECON == RECON_PLM) {
      lean_plm(Wm1, W0, Wp1, lo, up);
    } else if (FAST) {
      lean_ppm(Wm2, Wm1, W0, Wp1, Wp2, lo, up);
    } else {
      V5<R> l, u;
      reconstruct<RECON, false>(to_normal<D>(Wm2), to_normal<D>(Wm1), to_normal<D>(W0), to_normal<D>(Wp1), to_normal<D>(Wp2), p, l, u);
      lo = from_normal<D>(l);
      up = from_normal<D>(u);
    }
  }
  template <int D> static __device__ __forceinline__ V5<R> flux(const V5<R>& W, const Par<R>& p) {
    if (FAST) return lean_phys_flux<D>(W, p);
    return from_normal<D>(phys_flux(to_normal<D>(W), p));
  }
};

template <class R, int RECON, int RS, int FAST, int MINB, int GRID, int GC>
__global__ void __launch_bounds__(LEAN_NT, MINB)
mhm_lean_kernel(const R* __restrict__ in, R* __restrict__ out, R* __restrict__ face_flux, int Ng, int g_arg, Par<R> p,
                const R* __restrict__ max_speed, R cfl, long long* status, GridIO<R> gio) {
  using Op = LeanOps<R, RECON, RS, FAST>;
  using Mo = MhmOps<R, RECON, RS, FAST>;
  constexpr int GW = 2 + RECON, RW = 1 + RECON, SWP = PS + 2 * GW, WPL = SWP * SWP, NW = 2 * RW + 1, NPL = PS + 2 * GW;
  constexpr int NC = LEAN_COLS, NT = LEAN_NT, FT = PS + 2;
  apply_device_dt(p, max_speed, cfl);

  // ghost width: grid mode takes the ghost zones from the grid at the minimum width; GC >= 0: compiled in (strides fold into
  // immediate offsets)
  const int g = GRID ? GW : (GC >= 0 ? GC : g_arg);
  const int S = PS + 2 * g;
  const int SS = S * S;
  const size_t nS = (size_t)SS * S;
  const int off = g - GW;  // unused outer ghost layers
  // grid mode: plane / variable strides of the grids
  const size_t N2 = (size_t)(gio.Gy * PS) * (gio.Gx * PS), N3 = N2 * (gio.Gz * PS);

  extern __shared__ __align__(16) unsigned char smem[];
  uint64_t* bar = reinterpret_cast<uint64_t*>(smem);   // [2]
  // mbarriers [2] | ring: [NW] fields of WPL cells, the primitive planes t-RW .. t+RW | xy: [6] fields of NC cells, LOX UPX LOY
  // UPY FX FY | raw: [2][5][SS], the landing zone of the bulk copies (last: only its size depends on g)
  R* raw = reinterpret_cast<R*>(smem + 64) + NW * 5 * WPL + 6 * 5 * NC;
  // every shared-memory access below is LDS / STS [R + immediate] off 32-bit shared addresses formed once (hydro_ptx.cuh Fld<>);
  // the window base and tid are opaque so that ptxas holds them instead of re-deriving them (S2UR / S2R) at every use
  using FW = Fld<R, WPL>;  // a primitive plane of the ring
  using FC = Fld<R, NC>;   // an exchange field LOX .. FY
  constexpr uint32_t ES = sizeof(R), CF = FC::BYTES;
  uint32_t sb = smem_u32(smem);
  asm volatile("" : "+r"(sb));
  const uint32_t sm_ring = sb + 64u, sm_xy = sm_ring + (uint32_t)(NW * 5 * WPL) * ES, sm_raw = sm_xy + (uint32_t)(6 * 5 * NC) * ES;

  int tid = threadIdx.x;
  asm volatile("" : "+r"(tid));
  // warps 0-7: interior columns (two rows of 16 per warp); warp 8: x ring (i = -1, 16); warp 9: y ring (j = -1, 16)
  int ii, jj;
  if (tid < PS * PS) { jj = 1 + (tid >> 4); ii = 1 + (tid & 15); }
  else if (tid < PS * PS + 32) { const int l = tid - PS * PS; jj = 1 + (l >> 1); ii = (l & 1) ? FT - 1 : 0; }
  else { const int l = tid - PS * FT; jj = (l < PS) ? 0 : FT - 1; ii = 1 + (l & (PS - 1)); }
  const int col = jj * FT + ii;
  // the role is a property of the warp (0-7 interior, 8 the x ring, 9 the y ring): flags from a warp broadcast
  const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0);
  const bool in_i = warp != PS * PS / 32, in_j = warp != PS * PS / 32 + 1, interior = in_i && in_j;
  const int wb = (jj + GW - 1) * SWP + (ii + GW - 1);
  // per-thread addresses: own cell in ring slot 0 (vector part, scalar part at + dws), own column in LOX (cv, cs)
  const uint32_t w16 = sm_ring + 16u * (uint32_t)wb, dws = FW::SD - (16u - ES) * (uint32_t)wb;
  const uint32_t cv = sm_xy + 16u * (uint32_t)col, cs = cv + FC::SD - (16u - ES) * (uint32_t)col;
  uint32_t wo[NW];  // CTA-uniform byte offsets of the ring slots holding planes t-RW .. t+RW; rotate once per step
#pragma unroll
  for (int k = 0; k < NW; ++k) wo[k] = (uint32_t)k * FW::BYTES;
  const bool feeder = tid == PS * FT;  // lane 0 of the least loaded warp issues the bulk copies and waits for them

  const int my_groups = (Ng - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x;
  const int total_planes = my_groups * NPL;
  auto issue = [&](int n) {  // the feeder lane only
    asm volatile("" : "+r"(n));  // keeps the descriptor arithmetic inside the feeder's branch
    if (n >= total_planes) return;
    const int m = n / NPL, pl = n - m * NPL;
    const size_t grp = (size_t)blockIdx.x + (size_t)m * gridDim.x;
    const R* src = in + grp * 5 * nS + (size_t)(pl + off) * SS;
    uint64_t* b = bar + (n & 1);
    R* dst = raw + (size_t)(n & 1) * 5 * SS;
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
  GridFeed<R, SWP, NPL, NT> gf;
  gf.reset();
  if (GRID) { gf.feed(gio, my_groups, raw, tid); gf.feed(gio, my_groups, raw + 5 * WPL, tid); }
  else if (feeder) { issue(0); issue(1); }

  Cnt c = {0, 0, 0};
  typename Bits<R>::U best = 0;  // running maximum of the updated cells' wave speed (next_max_speed)
  int nseq = 0;
  // raw plane nseq has landed: grid mode: a thread waits for its own copies; batch mode: the feeder lane polls the mbarrier.
  // The CTA barrier that follows publishes the plane to all threads.
  auto landed = [&]() {
    if (GRID) cp_async_wait<1>();
    else if (feeder) mbar_wait(bar + (nseq & 1), (uint32_t)((nseq >> 1) & 1));
  };
  // con->prim of raw plane nseq into the ring slot at byte offset slot_off: cells tid and, for CR0 <= tid < CR2, tid + CSH
  // (CSH a whole number of plane rows: both cells of a thread share the column, one raw offset serves both)
  constexpr int CSH = (NT / SWP) * SWP, CR0 = NT - CSH, CR2 = WPL - CSH;
  uint32_t roff0;
  {
    const int b = tid / SWP, a = tid - b * SWP;
    roff0 = (uint32_t)((b + off) * S + (a + off)) * ES;
    asm volatile("" : "+r"(roff0));
  }
  auto convert = [&](uint32_t slot_off) {
    const uint32_t rp = sm_raw + (uint32_t)(nseq & 1) * (uint32_t)(5 * SS) * ES + roff0;
    const uint32_t dv = sm_ring + slot_off + 16u * (uint32_t)tid, ds = sm_ring + slot_off + FW::SD + ES * (uint32_t)tid;
    const uint32_t sS = (uint32_t)SS * ES;
    {
      V5<R> U;
#pragma unroll
      for (int q = 0; q < 5; ++q) U[q] = *sm_ptr<const R>(rp + (uint32_t)q * sS);
      FW::st(dv, ds, Op::c2p(U, p, c));
    }
    if (tid >= CR0 && tid < CR2) {
      const uint32_t rp1 = rp + (uint32_t)((CSH / SWP) * S) * ES;
      V5<R> U;
#pragma unroll
      for (int q = 0; q < 5; ++q) U[q] = *sm_ptr<const R>(rp1 + (uint32_t)q * sS);
      FW::st(dv + 16u * CSH, ds + ES * CSH, Op::c2p(U, p, c));
    }
  };
  auto refill = [&]() {
    if (GRID) gf.feed(gio, my_groups, raw + (size_t)(nseq & 1) * 5 * SS, tid);
    else if (feeder) { fence_async_smem(); issue(nseq + 2); }
    ++nseq;
  };

  V5<R> uzc, Dz;  // advanced up_z of plane t-1; (dF_x + dF_y) - F_z of plane t-1
#pragma unroll
  for (int q = 0; q < 5; ++q) { uzc[q] = R(0); Dz[q] = R(0); }

  for (int m = 0; m < my_groups; ++m) {
    const size_t grp = (size_t)blockIdx.x + (size_t)m * gridDim.x;
    // own cell of plane 0 in `in` / `out`, or (grid mode, interior columns) in the grids: plane stride SS / 256 or N2, variable stride nS / 4096 or N3
    const R* gin0 = in + grp * 5 * nS + ((size_t)g * S + (jj - 1 + g)) * S + (ii - 1 + g);
    R* gout0 = out + grp * 5 * PS * PS * PS + (jj - 1) * PS + (ii - 1);
    if (GRID) {
      const size_t cell = interior ? grid_cell0(gio, grp, ii - 1, jj - 1) : 0;
      gin0 = gio.gin + cell;
      gout0 = gio.gout + cell;
    }
    const size_t pstr_in = GRID ? N2 : (size_t)SS, vstr_in = GRID ? N3 : nS;
    R* gff = face_flux ? face_flux + grp * 9 * 5 * PS * PS : nullptr;
    for (int k = 0; k < NW; ++k) {  // prologue: planes -1-RW .. -1+RW
      landed();
      __syncthreads();
      convert(wo[k]);
      __syncthreads();
      refill();
    }

#pragma unroll 1
    for (int t = -1; t <= PS; ++t) {
      const bool tin = t >= 0 && t < PS;
      // ================= P1: face states of plane t, Hancock half step, F_z(t), update of plane t-1 =================
      if (tin || interior) {
        V5<R> Uold;
        const bool upd = interior && t >= 1;
        if (upd) {
          const R* gin = gin0 + (size_t)(t - 1) * pstr_in;
#pragma unroll
          for (int q = 0; q < 5; ++q) { Uold[q] = __ldg(gin); gin += vstr_in; }
        }
        const uint32_t w0 = w16 + wo[RW], s0 = w0 + dws;
        const V5<R> W0 = FW::ld(w0, s0);
        V5<R> lox, upx, loy, upy, loz, upz, inc;
        {
          const V5<R> Wb = FW::ld(w0 - 16u, s0 - ES), Wc = FW::ld(w0 + 16u, s0 + ES);
          V5<R> Wa = Wb, Wd = Wc;
          if (RECON == RECON_PPM) { Wa = FW::ld(w0 - 32u, s0 - 2 * ES); Wd = FW::ld(w0 + 32u, s0 + 2 * ES); }
          Mo::template recon<0>(Wa, Wb, W0, Wc, Wd, p, lox, upx);
          const V5<R> fu = Mo::template flux<0>(upx, p), fl = Mo::template flux<0>(lox, p);
#pragma unroll
          for (int q = 0; q < 5; ++q) inc[q] = fu[q] - fl[q];
        }
        {
          const V5<R> Wb = FW::ld(w0 - 16u * SWP, s0 - ES * SWP), Wc = FW::ld(w0 + 16u * SWP, s0 + ES * SWP);
          V5<R> Wa = Wb, Wd = Wc;
          if (RECON == RECON_PPM) { Wa = FW::ld(w0 - 32u * SWP, s0 - 2 * ES * SWP); Wd = FW::ld(w0 + 32u * SWP, s0 + 2 * ES * SWP); }
          Mo::template recon<1>(Wa, Wb, W0, Wc, Wd, p, loy, upy);
          const V5<R> fu = Mo::template flux<1>(upy, p), fl = Mo::template flux<1>(loy, p);
#pragma unroll
          for (int q = 0; q < 5; ++q) inc[q] = inc[q] + (fu[q] - fl[q]);
        }
        {
          const V5<R> Wb = FW::ld(w16 + wo[RW - 1], w16 + wo[RW - 1] + dws), Wc = FW::ld(w16 + wo[RW + 1], w16 + wo[RW + 1] + dws);
          V5<R> Wa = Wb, Wd = Wc;
          if (RECON == RECON_PPM) { Wa = FW::ld(w16 + wo[0], w16 + wo[0] + dws); Wd = FW::ld(w16 + wo[2 * RW], w16 + wo[2 * RW] + dws); }
          Mo::template recon<2>(Wa, Wb, W0, Wc, Wd, p, loz, upz);
          const V5<R> fu = Mo::template flux<2>(upz, p), fl = Mo::template flux<2>(loz, p);
#pragma unroll
          for (int q = 0; q < 5; ++q) inc[q] = p.hnu * (inc[q] + (fu[q] - fl[q]));
        }
        if (tin && in_j) {
          FC::st(cv + LF_LOX * CF, cs + LF_LOX * CF, Op::correct(lox, inc, p, c));
          FC::st(cv + LF_UPX * CF, cs + LF_UPX * CF, Op::correct(upx, inc, p, c));
        }
        if (tin && in_i) {
          FC::st(cv + LF_LOY * CF, cs + LF_LOY * CF, Op::correct(loy, inc, p, c));
          FC::st(cv + LF_UPY * CF, cs + LF_UPY * CF, Op::correct(upy, inc, p, c));
        }
        if (interior) {
          if (t >= 0) {
            const V5<R> Fz = Op::template riemann<2>(uzc, Op::correct(loz, inc, p, c), p, c);
            if (gff && (t & 7) == 0) st5(gff + (size_t)((6 + (t >> 3)) * 5) * 256 + (jj - 1) * PS + (ii - 1), 256, Fz);
            if (upd) {
              V5<R> U;
#pragma unroll
              for (int q = 0; q < 5; ++q) U[q] = Uold[q] - p.nu * (Dz[q] + Fz[q]);
              const V5<R> Wn = Op::c2p(U, p, c);
              if (p.next_speed) track_speed(Wn, p, best);
              if (!FAST && (p.min_dens > R(0) || p.min_pres > R(0))) U = prim2cons(Wn, p);
              if (GRID) {
                R* d = gout0 + (size_t)(t - 1) * N2;
#pragma unroll
                for (int q = 0; q < 5; ++q) { *d = U[q]; d += N3; }
              } else {
                st5(gout0 + (t - 1) * PS * PS, PS * PS * PS, U);
              }
            }
            Dz = Fz;
          }
          if (t < PS) uzc = Op::correct(upz, inc, p, c);
        }
      }
      const bool conv = t + RW + 1 <= PS - 1 + GW;  // plane t+RW+1 replaces plane t-RW (read for the last time in P1)
      if (conv) landed();
      __syncthreads();  // barrier A

      // ================= P2: F_x(t), F_y(t), boundary-flux stores; con->prim of the next plane =================
      if (tin) {
        if (in_j && ii >= 1) {
          const V5<R> f = Op::template riemann<0>(FC::ld(cv + LF_UPX * CF - 16u, cs + LF_UPX * CF - ES), FC::ld(cv + LF_LOX * CF, cs + LF_LOX * CF), p, c);
          FC::st(cv + LF_FX * CF, cs + LF_FX * CF, f);
          if (gff && ((ii - 1) & 7) == 0) st5(gff + (size_t)(((ii - 1) >> 3) * 5) * 256 + t * PS + (jj - 1), 256, f);
        }
        if (in_i && jj >= 1) {
          const V5<R> f = Op::template riemann<1>(FC::ld(cv + LF_UPY * CF - 16u * FT, cs + LF_UPY * CF - ES * FT), FC::ld(cv + LF_LOY * CF, cs + LF_LOY * CF), p, c);
          FC::st(cv + LF_FY * CF, cs + LF_FY * CF, f);
          if (gff && ((jj - 1) & 7) == 0) st5(gff + (size_t)((3 + ((jj - 1) >> 3)) * 5) * 256 + t * PS + (ii - 1), 256, f);
        }
      }
      if (conv) convert(wo[0]);
      __syncthreads();  // barrier B
      if (conv) refill();

      // ================= P3: carried x+y flux difference of plane t minus F_z(t) =================
      if (tin && interior) {
        const V5<R> x1 = FC::ld(cv + LF_FX * CF + 16u, cs + LF_FX * CF + ES), x0 = FC::ld(cv + LF_FX * CF, cs + LF_FX * CF);
        const V5<R> y1 = FC::ld(cv + LF_FY * CF + 16u * FT, cs + LF_FY * CF + ES * FT), y0 = FC::ld(cv + LF_FY * CF, cs + LF_FY * CF);
#pragma unroll
        for (int q = 0; q < 5; ++q) Dz[q] = ((x1[q] - x0[q]) + (y1[q] - y0[q])) - Dz[q];
      }
      {  // the ring slots rotate: the plane converted in P2 is now the newest
        const uint32_t w = wo[0];
#pragma unroll
        for (int k = 0; k + 1 < NW; ++k) wo[k] = wo[k + 1];
        wo[NW - 1] = w;
      }
    }
  }
  flush_counters(c, status);
  flush_speed(best, p.next_speed);
}

template <class R, int RECON, int RS, int FAST, int MINB, int GRID = 0, int GC = -1> cudaError_t launch_mhm_lean(const SolveArgs<R>& a) {
  // the default options at the ghost width of the AMR batches (g = 3) have their own fp32 instantiation (hydro_lean_ctu.cuh)
  if constexpr (FAST && !GRID && GC < 0 && sizeof(R) == 4) {
    if (a.g == 3) return launch_mhm_lean<R, RECON, RS, FAST, MINB, GRID, 3>(a);
  }
  auto kern = mhm_lean_kernel<R, RECON, RS, FAST, MINB, GRID, GC>;
  const size_t smem = mhm_smem_bytes(sizeof(R), RECON, a.g);
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
  e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, LEAN_NT, smem);
  if (e != cudaSuccess) return e;
  if (per_sm < 1) return cudaErrorInvalidConfiguration;
  long long grid = (long long)sms * per_sm;
  if (grid > a.Ng) grid = a.Ng;
  kern<<<(unsigned)grid, LEAN_NT, smem, a.stream>>>(a.in, a.out, a.face_flux, a.Ng, a.g, a.par, a.max_speed, a.cfl, a.status, a.grid);
  return cudaGetLastError();
}

}  // namespace hydro
