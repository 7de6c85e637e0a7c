// hydro_lean_ctu.cuh -- "lean" fused z-marching CTU kernel (steps (1)-(5) in one launch).
//
// Design point (from the ncu captures, profiles/): the path is bound by instruction ISSUE, not by HBM and not by the
// FMA pipe itself.  A column-per-thread z-march holds only 15 carried values per thread in registers; everything that
// crosses a phase boundary lives in shared memory, so that a 320-thread CTA fits in 96 registers and about 108 KB of
// shared memory (fp32, PLM) and TWO CTAs (two patch groups) are resident per SM, each hiding the other's barriers.
// Round 2 ("instruction diet", profiles/r2_*): packed FFMA2 was measured NOT to relieve the issue port on B200
// (profiles/r2_issue_probe.md), so the kernel instead strips everything that is not the method's arithmetic:
//   * every shared-memory access is `[R + immediate]` off per-thread 32-bit shared addresses formed once per kernel
//     (hydro_ptx.cuh Fld<>); the primitive-plane ring rotates by renaming three address registers;
//   * the three thread roles are separate code paths selected once per warp (warps 0-7 interior columns, warp 8 the
//     x ring, warp 9 the y ring), so that the interior path carries no role predicates;
//   * the Roe fallback crosses its call by value (no local memory anywhere: hydro_lean_math.cuh);
//   * one lane waits for the bulk copies and the next CTA barrier publishes them; the least loaded warp issues them.
//
// Thread -> column of the 18 x 18 tile (interior + one-cell ring): warps 0-7 own the 256 interior columns (two rows of
// 16 per warp), warp 8 the x ring (i = -1, 16) and warp 9 the y ring (j = -1, 16), which only do the work the ring
// needs.  The four corner columns only feed F*_x / F*_y of the ring; their work rides on lanes that would otherwise
// idle: their traced states are formed by 8 lanes of warp 9 during phase F of the previous step, their four first-pass
// Riemann problems by i = -1 lanes of warp 8 (F*_x) and j = -1 lanes of warp 9 (F*_y) in phase D.
//
// Step t = -2 .. 16 of a group (plane index; W = primitive planes in a ring, one plane converted per step):
//   B  z: traced states of plane t+1 (own column of the ring planes) -> private slots;
//         F*_z(t+1) = RS(up_z(t), lo_z(t+1)); dF*_z(t) kept in registers
//   C  x,y: traced states of plane t -> LOX, UPX, LOY, UPY                                  | barrier 1
//   D  F*_x(t), F*_y(t) -> FX, FY;  con->prim of the next raw plane into the ring           | barrier 2
//   E  transverse correction (half nu, S4) of the x,y states in place and of the z states;
//      F_z(t) = RS(up_z'(t-1), lo_z'(t)); conservative update + store of plane t-1          | barrier 3
//   F  F_x(t), F_y(t) -> FX, FY; patch-boundary flux stores; corner states of plane t+1     | barrier 4
//   G  carried D_z = (dF_x + dF_y)(t) - F_z(t), so that the update is U - nu (D_z + F_z(t+1))
// Input planes arrive by 1-D bulk async copies (cp.async.bulk + mbarrier), two planes in flight, running
// ahead across group boundaries.
#pragma once
#include <cstdint>
#include "hydro_launch.cuh"
#include "hydro_lean_math.cuh"
#include "hydro_ptx.cuh"

namespace hydro {

#ifndef LEAN_ROLE_SPLIT
#define LEAN_ROLE_SPLIT 0
#endif
#ifndef LEAN_OPAQUE
#define LEAN_OPAQUE 1
#endif
#ifndef LEAN_GC_F64
#define LEAN_GC_F64 0  // measured: the fp64 kernel (ten warps per SM, latency-bound) is 3 % slower with it despite 2 % fewer instructions
#endif
#ifndef LEAN_ONE_WAITER
#define LEAN_ONE_WAITER 1  // 1: one lane polls the plane's mbarrier before barrier 1; 0: every thread polls it in phase D
#endif
enum : int { LF_LOX = 0, LF_UPX, LF_LOY, LF_UPY, LF_FX, LF_FY };
enum : int { ROLE_INT = 0, ROLE_XR = 1, ROLE_YR = 2, ROLE_ANY = 3 };  // ROLE_ANY: one code stream, roles decided at run time

// variant seams: FAST = van Leer limiter on primitive variables, no floors (compile time)
template <class R, int RECON, int RS, int FAST> struct LeanOps {
  static __device__ __forceinline__ V5<R> c2p(const V5<R>& U, const Par<R>& p, Cnt& c) {
    if (FAST) return lean_cons2prim(U, p, c.bad);
    return cons2prim(U, p, c);
  }
  static __device__ __forceinline__ V5<R> correct(const V5<R>& W, const V5<R>& dq, const Par<R>& p, Cnt& c) {
    if (FAST) return lean_correct(W, dq, p, c.bad);
    V5<R> U = prim2cons(W, p);
#pragma unroll
    for (int q = 0; q < 5; ++q) U[q] = U[q] - dq[q];
    return cons2prim(U, p, c);
  }
  // traced face states of the middle cell of a normal-frame pencil
  static __device__ __forceinline__ void recon(const V5<R>& Wm2, const V5<R>& Wm1, const V5<R>& W0, const V5<R>& Wp1,
                                               const V5<R>& Wp2, const Par<R>& p, V5<R>& lo, V5<R>& up) {
    if (FAST && RECON == RECON_PLM) lean_plm_trace(Wm1, W0, Wp1, p, p.nu, p.hnu, lo, up);
    else if (FAST) lean_ppm_trace(Wm2, Wm1, W0, Wp1, Wp2, p, p.nu, lo, up);
    else reconstruct<RECON, true>(Wm2, Wm1, W0, Wp1, Wp2, p, lo, up);
  }
  // trackers of non-positive states other than the per-conversion count (hydro_lean_math.cuh BadMin)
  template <class T> static __device__ __forceinline__ V5<R> c2p(const V5<R>& U, const Par<R>& p, Cnt& c, T& trk) {
    if (FAST) return lean_cons2prim(U, p, trk);
    return cons2prim(U, p, c);
  }
  template <class T> static __device__ __forceinline__ V5<R> correct(const V5<R>& W, const V5<R>& dq, const Par<R>& p, Cnt& c, T& trk) {
    if (FAST) return lean_correct(W, dq, p, trk);
    return correct(W, dq, p, c);
  }
  // the flux times `scale` (the CTU first pass wants nu/2 F*: free inside the lean Roe solver)
  template <int D> static __device__ __forceinline__ V5<R> riemann_scaled(const V5<R>& WL, const V5<R>& WR, const Par<R>& p, Cnt& c, R scale) {
    if (FAST && RS == RS_ROE) return from_normal<D>(lean_roe_scaled(to_normal<D>(WL), to_normal<D>(WR), p, c, scale));
    V5<R> F = riemann<D>(WL, WR, p, c);
#pragma unroll
    for (int q = 0; q < 5; ++q) F[q] = scale * F[q];
    return F;
  }
  template <int D> static __device__ __forceinline__ V5<R> riemann(const V5<R>& WL, const V5<R>& WR, const Par<R>& p, Cnt& c) {
    const V5<R> l = to_normal<D>(WL), r = to_normal<D>(WR);
    if (FAST && RS == RS_ROE) return from_normal<D>(lean_roe(l, r, p, c));
    if (FAST && RS == RS_HLLC) return from_normal<D>(lean_hllc(l, r, p));
    if (FAST && RS == RS_EXACT) return from_normal<D>(lean_exact(l, r, p, c));
    if (FAST && RS == RS_HLLE) return from_normal<D>(lean_hlle(l, r, p));
    return from_normal<D>(riemann_n<RS>(l, r, p, c));
  }
};

// what a role needs from the kernel prologue: pointers, geometry, shared-memory bases
template <class R> struct LeanCtx {
  const R* in; R* out; R* face_flux;
  int Ng, g;
  long long* status;
  GridIO<R> gio;
  uint32_t sm_bar, sm_ring, sm_zs, sm_xy, sm_raw;  // shared-space byte addresses
  uint64_t* bar;
  R* raw;
};

// The whole march of one role over this CTA's groups.  All roles execute the same sequence of CTA barriers.
template <class R, int RECON, int RS, int FAST, int GRID, int ROLE, int GC>
__device__ __forceinline__ void ctu_lean_role(const LeanCtx<R>& cx, const Par<R>& p, int ii, int jj, const int tid) {
  using Op = LeanOps<R, RECON, RS, FAST>;
  constexpr int GW = 2 + RECON, RW = 1 + RECON, SWP = PS + 2 * GW, WPL = SWP * SWP, NW = 2 * RW + 1, NPL = PS + 2 * GW;
  // PPM tiles are trimmed so that two fp32 CTAs (or one fp64 CTA) fit: one raw landing plane instead of two, and the
  // oldest plane of the z pencil (needed only at the thread's own column) carried in registers instead of the ring
  constexpr int NRAW = RECON == RECON_PPM ? 1 : 2, RC = RECON == RECON_PPM ? 1 : 0, NWS = NW - RC;  // == LEAN_NRAW, LEAN_RING_CARRY
  constexpr int NC = LEAN_COLS, NT = LEAN_NT, FT = PS + 2;
  constexpr uint32_t ES = sizeof(R);
  using FW = Fld<R, WPL>;  // a primitive plane of the ring
  using FZ = Fld<R, NT>;   // a private traced-z field (one entry per thread)
  using FC = Fld<R, NC>;   // an exchange field LOX .. FY (one entry per column)
  // the column lies inside the interior range along x / y; with ROLE_ANY these are run-time flags of one code stream
  // (three specialised streams cost more in instruction-cache misses than they save: profiles/r2_ctu_diet.md)
#if LEAN_OPAQUE
  // the role is a property of the WARP (warps 0-7 interior, 8 the x ring, 9 the y ring): taken from a warp broadcast, the
  // flags are uniform values and every role test is a uniform branch (no BSSY / BSYNC, no per-lane predicate re-derived
  // from tid at each use)
  const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0);
  const bool in_i = ROLE == ROLE_ANY ? (warp != PS * PS / 32) : ROLE != ROLE_XR;
  const bool in_j = ROLE == ROLE_ANY ? (warp != PS * PS / 32 + 1) : ROLE != ROLE_YR;
#else
  const bool in_i = ROLE == ROLE_ANY ? (ii >= 1 && ii <= PS) : ROLE != ROLE_XR;
  const bool in_j = ROLE == ROLE_ANY ? (jj >= 1 && jj <= PS) : ROLE != ROLE_YR;
#endif
  const bool INT = in_i && in_j, XR = !in_i, YR = !in_j;

  // ghost width: a compile-time constant in the specialised instantiations (GC >= 0; grid mode: always GW), so that plane and
  // variable strides fold into immediate offsets
  const int g = GRID ? GW : (GC >= 0 ? GC : cx.g);
  const int S = PS + 2 * g;
  const int SS = S * S;
  const size_t nS = (size_t)SS * S;
  const int off = g - GW;  // unused outer ghost layers (grid mode: g == GW)
  const GridIO<R>& gio = cx.gio;
  // grid mode: cells per axis, plane / variable strides of the grids, boundary folding
  const int Nx = gio.Gx * PS, Ny = gio.Gy * PS, Nz = gio.Gz * PS;
  const size_t N2 = (size_t)Ny * Nx, N3 = N2 * Nz;
  auto fold = [&](int c, int N) {
    return gio.bc == 0 ? (c < 0 ? c + N : (c >= N ? c - N : c)) : (c < 0 ? 0 : (c >= N ? N - 1 : c));
  };

  const int col = jj * FT + ii;
  const int wb = (jj + GW - 1) * SWP + (ii + GW - 1);  // own index in a primitive plane
  // ---- per-thread shared addresses (vector part; the scalar part of the same cell sits at + d?s)
  // own cell in the ring slots, oldest plane first: a per-thread base plus CTA-uniform slot offsets that rotate once per step
  // (the rotation state lives in uniform registers; per-thread rotating addresses cost three more live registers)
  const uint32_t w16 = cx.sm_ring + 16u * (uint32_t)wb;
  uint32_t wo[NWS];
#pragma unroll
  for (int k = 0; k < NWS; ++k) wo[k] = (uint32_t)k * FW::BYTES;
#define wv(k) (w16 + wo[k])
  const uint32_t dws = FW::SD - (16u - ES) * (uint32_t)wb;
  const uint32_t z16 = cx.sm_zs + 16u * (uint32_t)tid;
  uint32_t zo = 0;                                           // uniform: parity slot [lo, up] read this step (the other is written)
#define zcur (z16 + zo)
#define znxt (z16 + (2u * FZ::BYTES - zo))
  const uint32_t dzs = FZ::SD - (16u - ES) * (uint32_t)tid;
  const uint32_t cv = cx.sm_xy + 16u * (uint32_t)col;
  const uint32_t cs = cv + FC::SD - (16u - ES) * (uint32_t)col;
  constexpr uint32_t CF = FC::BYTES;  // bytes per exchange field
  // first-pass face jobs of phase D: own lower faces, plus (ring roles) the corner faces on lanes that have none
  int fxc = (INT || ii >= 1) ? col : -1, fyc = (INT || jj >= 1) ? col : -1;
  if (XR) {
    if (ii == 0 && jj == 1) fxc = FT - 1;               // F*_x(f = 16, j = -1)
    if (ii == 0 && jj == 2) fxc = FT * FT - 1;          // F*_x(f = 16, j = 16)
  }
  if (YR) {
    if (jj == 0 && ii == 1) fyc = (FT - 1) * FT;        // F*_y(i = -1, f = 16)
    if (jj == 0 && ii == 2) fyc = FT * FT - 1;          // F*_y(i = 16, f = 16)
  }
  const uint32_t fxv = cx.sm_xy + 16u * (uint32_t)fxc, fxs = fxv + FC::SD - (16u - ES) * (uint32_t)fxc;
  const uint32_t fyv = cx.sm_xy + 16u * (uint32_t)fyc, fys = fyv + FC::SD - (16u - ES) * (uint32_t)fyc;
  // corner-state job of phase F: lanes 0..7 of warp 9: corner (l & 3), direction (l >> 2)
  const int cl = tid - PS * FT;
  const bool cjob = YR && cl >= 0 && cl < 8;
  const int cdir = (cl >> 2) & 1;
  const int cci = (cl & 1) ? FT - 1 : 0, ccj = (cl & 2) ? FT - 1 : 0;
  const int ccol = ccj * FT + cci, cwb = (ccj + GW - 1) * SWP + (cci + GW - 1);
  // the bulk copies are issued, and waited for, by one lane of the least loaded warp (warp 9, the y ring)
  const bool feeder = YR && tid == PS * FT;

  // ---- plane pipeline: sequence number n = m * NPL + (plane + GW) over this CTA's groups m
  const int my_groups = (cx.Ng - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x;
  const int total_planes = my_groups * NPL;
  auto issue = [&](int n) {  // the feeder lane only
#if LEAN_OPAQUE
    asm volatile("" : "+r"(n));  // keeps the descriptor arithmetic below inside the feeder's branch (hoisted, every warp would run it)
#endif
    if (n >= total_planes) return;
    const int m = n / NPL, pl = n - m * NPL;
    const size_t grp = (size_t)blockIdx.x + (size_t)m * gridDim.x;
    const R* src = cx.in + grp * 5 * nS + (size_t)(pl + off) * SS;
    uint64_t* b = cx.bar + (n % NRAW);
    R* dst = cx.raw + (size_t)(n % NRAW) * 5 * SS;
    mbar_expect_tx(b, (uint32_t)(5 * SS * sizeof(R)));
#pragma unroll
    for (int q = 0; q < 5; ++q) bulk_g2s(dst + (size_t)q * SS, src + q * nS, (uint32_t)(SS * sizeof(R)), b);
  };
  // grid mode: every thread copies its share of raw plane n (element-wise async copies, ghost cells folded).  Planes are
  // fed strictly in sequence, so the (group, plane) of the next feed is running state, not a division of n.
  // (A variant with padded raw rows and 16-byte copies of the aligned interior cells measured 15 % slower.)
  int f_pl = 0, f_m = 0, f_g = 0;  // plane within the group, group counter of this CTA, packed group coordinates (10 bits each)
  auto feed = [&](int n) {
    if (f_m < my_groups) {
      if (f_pl == 0) {
        const int grp = (int)blockIdx.x + f_m * (int)gridDim.x;
        f_g = (grp % gio.Gx) | (((grp / gio.Gx) % gio.Gy) << 10) | ((grp / (gio.Gx * gio.Gy)) << 20);
      }
      const int x0 = (f_g & 1023) * PS - GW, y0 = ((f_g >> 10) & 1023) * PS - GW, z0 = (f_g >> 20) * PS - GW;
      const R* zsrc = gio.gin + (size_t)fold(z0 + f_pl, Nz) * N2;
      R* dst = cx.raw + (size_t)(n % NRAW) * 5 * (SWP * SWP);
#pragma unroll
      for (int r = 0; r < (SWP * SWP + NT - 1) / NT; ++r) {
        const int pos = tid + r * NT;
        if (pos < SWP * SWP) {
          const int j = pos / SWP, i = pos - j * SWP;  // grid mode: S == SWP, a compile-time constant
          const R* sp = zsrc + (size_t)fold(y0 + j, Ny) * Nx + fold(x0 + i, Nx);
#pragma unroll
          for (int q = 0; q < 5; ++q) { cp_async_elem(dst + q * (SWP * SWP) + pos, sp); sp += N3; }
        }
      }
      if (++f_pl == NPL) { f_pl = 0; ++f_m; }
    }
    cp_async_commit();  // also when empty: keeps the wait_group arithmetic uniform
  };
  if (GRID) { feed(0); if (NRAW > 1) feed(1); }
  else if (feeder) { issue(0); if (NRAW > 1) issue(1); }

  Cnt c = {0, 0, 0};
  typename BadTrk<R>::type trk;  // non-positive rho / P seen by the conversions of this step (flushed into c.bad once per step)
  trk_reset(trk);
  typename Bits<R>::U best = 0;  // running maximum of the updated cells' wave speed (next_max_speed)
  int nseq = 0;  // planes converted so far
  // the raw plane the next conversion reads has landed: one lane polls the mbarrier (grid mode: every thread waits for its
  // own copies); the CTA barrier that follows publishes the plane to all threads
  auto landed = [&]() {
    if (GRID) cp_async_wait<NRAW - 1>();
    else if (LEAN_ONE_WAITER && feeder) mbar_wait(cx.bar + (nseq % NRAW), (uint32_t)((nseq / NRAW) & 1));
  };
  // prologue form: no barrier follows before the conversion, so every thread observes the mbarrier itself
  auto landed_all = [&]() {
    if (GRID) { cp_async_wait<NRAW - 1>(); __syncthreads(); }
    else mbar_wait(cx.bar + (nseq % NRAW), (uint32_t)((nseq / NRAW) & 1));
  };
  // con->prim of the next raw plane into the ring slot whose own-cell address is wslot (all threads; cells tid and, for the
  // first CR2 threads from CR0 on, tid + CSH: CSH is a whole number of plane rows, so that both cells of a thread share the
  // column and the raw offset of the second is the first's plus a uniform constant)
  constexpr int CSH = (NT / SWP) * SWP, CR0 = NT - CSH, CR2 = WPL - CSH;  // PLM: 320, 0, 80; PPM: 308, 12, 176
  uint32_t roff0;                                             // byte offset of cell tid in a raw plane (per variable: + q SS)
  {
    const int b = tid / SWP, a = tid - b * SWP;
    roff0 = (uint32_t)((b + off) * S + (a + off)) * ES;
#if LEAN_OPAQUE
    asm volatile("" : "+r"(roff0));
#endif
  }
  // Destination: cell tid of a ring slot sits at (z16, z16 + dzs) -- the thread's own z-state entry -- plus the compile-time
  // distance between the two arrays plus the slot's CTA-uniform offset: no per-thread address is formed for it.
  constexpr uint32_t RZV = (uint32_t)(NWS * 5 * WPL) * ES;               // sm_zs - sm_ring
  auto convert = [&](uint32_t slot_off) {
    const uint32_t rp = cx.sm_raw + (uint32_t)(nseq % NRAW) * (uint32_t)(5 * SS) * ES + roff0;
    const uint32_t dv = z16 + slot_off - RZV, ds = dv + dzs + (FW::SD - FZ::SD);
    const uint32_t sS = (uint32_t)SS * ES;
    {
      V5<R> U;
#pragma unroll
      for (int q = 0; q < 5; ++q) U[q] = *sm_ptr<const R>(rp + (uint32_t)q * sS);
      FW::st(dv, ds, Op::c2p(U, p, c, trk));
    }
    if (tid >= CR0 && tid < CR2) {
      const uint32_t rp1 = rp + (uint32_t)((CSH / SWP) * S) * ES;
      V5<R> U;
#pragma unroll
      for (int q = 0; q < 5; ++q) U[q] = *sm_ptr<const R>(rp1 + (uint32_t)q * sS);
      FW::st(dv + 16u * CSH, ds + ES * CSH, Op::c2p(U, p, c, trk));
    }
  };
  // after the barrier that follows a conversion: refill the raw stage it consumed
  auto refill = [&]() {
    if (GRID) feed(nseq + NRAW);
    else if (feeder) { fence_async_smem(); issue(nseq + NRAW); }
    ++nseq;
  };
  // traced states of a corner column of the primitive plane in slot `wslot` along x (cdir 0) or y (cdir 1)
  auto corner_states = [&](uint32_t wslot) {
    const int st = cdir ? SWP : 1;
    const uint32_t base = wslot - 16u * (uint32_t)wb;
    V5<R> W[2 * RW + 1];
#pragma unroll
    for (int s = 0; s < 2 * RW + 1; ++s) {
      const uint32_t i = (uint32_t)(cwb + (s - RW) * st);
      const V5<R> w = FW::ld(base + 16u * i, base + FW::SD + ES * i);
      W[s][0] = w[0]; W[s][4] = w[4];
      W[s][1] = cdir ? w[2] : w[1];
      W[s][2] = cdir ? w[3] : w[2];
      W[s][3] = cdir ? w[1] : w[3];
    }
    V5<R> l, u, lo, up;
    Op::recon(W[0], W[RW - 1], W[RW], W[RW + 1], W[2 * RW], p, l, u);
    lo[0] = l[0]; lo[4] = l[4]; up[0] = u[0]; up[4] = u[4];
    lo[1] = cdir ? l[3] : l[1]; up[1] = cdir ? u[3] : u[1];
    lo[2] = cdir ? l[1] : l[2]; up[2] = cdir ? u[1] : u[2];
    lo[3] = cdir ? l[2] : l[3]; up[3] = cdir ? u[2] : u[3];
    const uint32_t v = cx.sm_xy + 16u * (uint32_t)ccol + (uint32_t)(2 * cdir) * CF, s = cx.sm_xy + FC::SD + ES * (uint32_t)ccol + (uint32_t)(2 * cdir) * CF;
    FC::st(v + LF_LOX * CF, s + LF_LOX * CF, lo);
    FC::st(v + LF_UPX * CF, s + LF_UPX * CF, up);
  };

  V5<R> f1z, uzc, Dz;  // F*_z at the lower face of plane t+1; corrected up_z of plane t-1; (dF_x + dF_y) - F_z of plane t-1
#pragma unroll
  for (int q = 0; q < 5; ++q) { f1z[q] = R(0); uzc[q] = R(0); Dz[q] = R(0); }

  for (int m = 0; m < my_groups; ++m) {
    const size_t grp = (size_t)blockIdx.x + (size_t)m * gridDim.x;
    // own cell of plane -1 in `in` / `out` (interior columns only); both advance by one plane per step from t = 0 on
    const R* gin = cx.in;
    R* gout = cx.out;
    R* gff = nullptr;
    if (INT) {
      gin = cx.in + grp * 5 * nS + ((size_t)(g - 1) * S + (jj - 1 + g)) * S + (ii - 1 + g);
      gout = cx.out + grp * 5 * PS * PS * PS + (jj - 1) * PS + (ii - 1) - PS * PS;
      if (GRID) {  // U^n and the result live in the grids: plane stride N2, variable stride N3
        const int gi = (int)grp, gx = gi % gio.Gx, gy = (gi / gio.Gx) % gio.Gy, gz = gi / (gio.Gx * gio.Gy);
        const size_t cell = ((size_t)(gz * PS) * Ny + gy * PS + (jj - 1)) * Nx + gx * PS + (ii - 1);
        gin = gio.gin + cell - N2;
        gout = gio.gout + cell - N2;
      }
    }
    gff = cx.face_flux ? cx.face_flux + grp * 9 * 5 * PS * PS : nullptr;
    // ---- prologue: the first NW primitive planes (-GW .. -GW+NW-1)
    V5<R> Wold;  // RC: W(t+1-RW) at the thread's own column
    if (RC) {
      landed_all();
      convert(wo[0]);
      __syncthreads();
      refill();
      Wold = FW::ld(wv(0), wv(0) + dws);
      __syncthreads();
    }
#pragma unroll
    for (int k = 0; k < NWS; ++k) {
      landed_all();
      convert(wo[k]);
      __syncthreads();
      refill();
    }

#pragma unroll 1
    for (int t = -2; t <= PS; ++t) {
      const bool doxy = t >= -1;
      const bool tin = t >= 0 && t < PS;
      // ================= B: z states of plane t+1, F*_z(t+1) =================
      V5<R> dFz;
#pragma unroll
      for (int q = 0; q < 5; ++q) dFz[q] = R(0);
      if (t < PS) {
        V5<R> Wz[NW];
#pragma unroll
        for (int s = RC; s < NW; ++s) {
          const V5<R> w = FW::ld(wv(s - RC), wv(s - RC) + dws);
          if (RC && s == RC) { Wz[0] = to_normal<2>(Wold); Wold = w; }
          Wz[s] = to_normal<2>(w);
        }
        V5<R> l, u;
        Op::recon(Wz[0], Wz[RW - 1], Wz[RW], Wz[RW + 1], Wz[2 * RW], p, l, u);
        const V5<R> lz = from_normal<2>(l), uz = from_normal<2>(u);
        FZ::st(znxt, znxt + dzs, lz);
        FZ::st(znxt + FZ::BYTES, znxt + FZ::BYTES + dzs, uz);
        if (t >= -1) {
          const V5<R> uzp = FZ::ld(zcur + FZ::BYTES, zcur + FZ::BYTES + dzs);
          const V5<R> f = Op::template riemann_scaled<2>(uzp, lz, p, c, p.hnu);  // nu/2 F*_z
#pragma unroll
          for (int q = 0; q < 5; ++q) { dFz[q] = f[q] - f1z[q]; f1z[q] = f[q]; }
        }
      }
      // ================= C: x,y traced states of plane t (slot RW-1 of the held planes) =================
      if (doxy) {
        const uint32_t w0 = wv(RW - 1 - RC), s0 = w0 + dws;
        const V5<R> W0 = FW::ld(w0, s0);
        {
          const V5<R> Wb = FW::ld(w0 - 16u, s0 - ES), Wc = FW::ld(w0 + 16u, s0 + ES);
          V5<R> Wa = Wb, Wd = Wc;
          if (RECON == RECON_PPM) { Wa = FW::ld(w0 - 32u, s0 - 2 * ES); Wd = FW::ld(w0 + 32u, s0 + 2 * ES); }
          V5<R> l, u;
          Op::recon(to_normal<0>(Wa), to_normal<0>(Wb), to_normal<0>(W0), to_normal<0>(Wc), to_normal<0>(Wd), p, l, u);
          FC::st(cv + LF_LOX * CF, cs + LF_LOX * CF, from_normal<0>(l));
          FC::st(cv + LF_UPX * CF, cs + LF_UPX * CF, from_normal<0>(u));
        }
        {
          const V5<R> Wb = FW::ld(w0 - 16u * SWP, s0 - ES * SWP), Wc = FW::ld(w0 + 16u * SWP, s0 + ES * SWP);
          V5<R> Wa = Wb, Wd = Wc;
          if (RECON == RECON_PPM) { Wa = FW::ld(w0 - 32u * SWP, s0 - 2 * ES * SWP); Wd = FW::ld(w0 + 32u * SWP, s0 + 2 * ES * SWP); }
          V5<R> l, u;
          Op::recon(to_normal<1>(Wa), to_normal<1>(Wb), to_normal<1>(W0), to_normal<1>(Wc), to_normal<1>(Wd), p, l, u);
          FC::st(cv + LF_LOY * CF, cs + LF_LOY * CF, from_normal<1>(l));
          FC::st(cv + LF_UPY * CF, cs + LF_UPY * CF, from_normal<1>(u));
        }
      }
      const bool conv = t + 2 + RW <= PS - 1 + GW;  // plane t+2+RW replaces plane t+1-RW (read for the last time in B / C)
      if (conv) landed();  // the raw plane converted in D (the barrier publishes it)
      __syncthreads();  // barrier 1

      // ================= D: F*_x(t), F*_y(t); con->prim of the next plane =================
      if (doxy) {
        if (INT || fxc >= 0)
          FC::st(fxv + LF_FX * CF, fxs + LF_FX * CF,
                 Op::template riemann_scaled<0>(FC::ld(fxv + LF_UPX * CF - 16u, fxs + LF_UPX * CF - ES), FC::ld(fxv + LF_LOX * CF, fxs + LF_LOX * CF), p, c, p.hnu));
        if (INT || fyc >= 0)
          FC::st(fyv + LF_FY * CF, fys + LF_FY * CF,
                 Op::template riemann_scaled<1>(FC::ld(fyv + LF_UPY * CF - 16u * FT, fys + LF_UPY * CF - ES * FT), FC::ld(fyv + LF_LOY * CF, fys + LF_LOY * CF), p, c, p.hnu));
      }
      if (!LEAN_ONE_WAITER && !GRID && conv) mbar_wait(cx.bar + (nseq % NRAW), (uint32_t)((nseq / NRAW) & 1));
      if (conv) convert(wo[0]);  // the oldest shared-memory plane: last read in B / C of this step
      __syncthreads();  // barrier 2
      if (conv) refill();

      // ================= E: transverse correction, F_z(t), update of plane t-1 =========
      if (doxy) {
        V5<R> Uold;
        const bool upd = INT && t >= 1;
        if (upd) {
          const R* gp = gin;
#pragma unroll
          for (int q = 0; q < 5; ++q) { Uold[q] = __ldg(gp); gp += GRID ? N3 : nS; }
        }
        V5<R> dFx, dFy;
#pragma unroll
        for (int q = 0; q < 5; ++q) { dFx[q] = R(0); dFy[q] = R(0); }
        if (in_i) {
          const V5<R> a = FC::ld(cv + LF_FX * CF + 16u, cs + LF_FX * CF + ES), b = FC::ld(cv + LF_FX * CF, cs + LF_FX * CF);
#pragma unroll
          for (int q = 0; q < 5; ++q) dFx[q] = a[q] - b[q];
        }
        if (in_j) {
          const V5<R> a = FC::ld(cv + LF_FY * CF + 16u * FT, cs + LF_FY * CF + ES * FT), b = FC::ld(cv + LF_FY * CF, cs + LF_FY * CF);
#pragma unroll
          for (int q = 0; q < 5; ++q) dFy[q] = a[q] - b[q];
        }
        if (tin && in_j) {  // x states: t1 = y, t2 = z
          V5<R> dq;
#pragma unroll
          for (int q = 0; q < 5; ++q) dq[q] = dFy[q] + dFz[q];  // the first-pass fluxes carry the factor nu/2
          FC::st(cv + LF_LOX * CF, cs + LF_LOX * CF, Op::correct(FC::ld(cv + LF_LOX * CF, cs + LF_LOX * CF), dq, p, c, trk));
          FC::st(cv + LF_UPX * CF, cs + LF_UPX * CF, Op::correct(FC::ld(cv + LF_UPX * CF, cs + LF_UPX * CF), dq, p, c, trk));
        }
        if (tin && in_i) {  // y states: t1 = z, t2 = x
          V5<R> dq;
#pragma unroll
          for (int q = 0; q < 5; ++q) dq[q] = dFz[q] + dFx[q];
          FC::st(cv + LF_LOY * CF, cs + LF_LOY * CF, Op::correct(FC::ld(cv + LF_LOY * CF, cs + LF_LOY * CF), dq, p, c, trk));
          FC::st(cv + LF_UPY * CF, cs + LF_UPY * CF, Op::correct(FC::ld(cv + LF_UPY * CF, cs + LF_UPY * CF), dq, p, c, trk));
        }
        if (INT) {  // z states: t1 = x, t2 = y; every plane t in [-1,16]
          V5<R> dq;
#pragma unroll
          for (int q = 0; q < 5; ++q) dq[q] = dFx[q] + dFy[q];
          if (t >= 0) {
            const V5<R> lzc = Op::correct(FZ::ld(zcur, zcur + dzs), dq, p, c, trk);
            const V5<R> Fz = Op::template riemann<2>(uzc, lzc, p, c);
            if (gff && (t & 7) == 0)  // stored right after the solve
              st5(gff + (size_t)((6 + (t >> 3)) * 5) * 256 + (jj - 1) * PS + (ii - 1), 256, Fz);
            if (upd) {
              V5<R> U;
#pragma unroll
              for (int q = 0; q < 5; ++q) U[q] = Uold[q] - p.nu * (Dz[q] + Fz[q]);
              const V5<R> Wn = Op::c2p(U, p, c, trk);
              if (p.next_speed) track_speed(Wn, p, best);
              if (!FAST && (p.min_dens > R(0) || p.min_pres > R(0))) U = prim2cons(Wn, p);
              if (GRID) {
                R* d = gout;
#pragma unroll
                for (int q = 0; q < 5; ++q) { *d = U[q]; d += N3; }
              } else {
                st5(gout, PS * PS * PS, U);
              }
            }
            Dz = Fz;
          }
          if (t < PS) uzc = Op::correct(FZ::ld(zcur + FZ::BYTES, zcur + FZ::BYTES + dzs), dq, p, c, trk);
        }
      }
      __syncthreads();  // barrier 3

      // ================= F: final fluxes of plane t + boundary-flux store ============
      if (tin) {
        if (in_j && (INT || ii >= 1)) {
          const V5<R> f = Op::template riemann<0>(FC::ld(cv + LF_UPX * CF - 16u, cs + LF_UPX * CF - ES), FC::ld(cv + LF_LOX * CF, cs + LF_LOX * CF), p, c);
          FC::st(cv + LF_FX * CF, cs + LF_FX * CF, f);
          if (gff && ((ii - 1) & 7) == 0) st5(gff + (size_t)(((ii - 1) >> 3) * 5) * 256 + t * PS + (jj - 1), 256, f);
        }
        if (in_i && (INT || jj >= 1)) {
          const V5<R> f = Op::template riemann<1>(FC::ld(cv + LF_UPY * CF - 16u * FT, cs + LF_UPY * CF - ES * FT), FC::ld(cv + LF_LOY * CF, cs + LF_LOY * CF), p, c);
          FC::st(cv + LF_FY * CF, cs + LF_FY * CF, f);
          if (gff && ((jj - 1) & 7) == 0) st5(gff + (size_t)((3 + ((jj - 1) >> 3)) * 5) * 256 + t * PS + (ii - 1), 256, f);
        }
      }
      // corner columns of plane t+1 (held in ring slot RW); their entries of LOX..UPY were last read in D
      if (YR && cjob && t < PS) corner_states(wv(RW - RC));
      __syncthreads();  // barrier 4

      // ================= G: carried x+y flux difference of plane t minus F_z(t) =================
      if (INT && tin) {
        const V5<R> x1 = FC::ld(cv + LF_FX * CF + 16u, cs + LF_FX * CF + ES), x0 = FC::ld(cv + LF_FX * CF, cs + LF_FX * CF);
        const V5<R> y1 = FC::ld(cv + LF_FY * CF + 16u * FT, cs + LF_FY * CF + ES * FT), y0 = FC::ld(cv + LF_FY * CF, cs + LF_FY * CF);
#pragma unroll
        for (int q = 0; q < 5; ++q) Dz[q] = ((x1[q] - x0[q]) + (y1[q] - y0[q])) - Dz[q];
      }
      // next step: the ring slots rotate (the converted plane is now the newest), the z-state slots swap, U^n / out advance
      {
        const uint32_t w = wo[0];
#pragma unroll
        for (int k = 0; k + 1 < NWS; ++k) wo[k] = wo[k + 1];
        wo[NWS - 1] = w;
        zo = 2u * FZ::BYTES - zo;
        c.bad += trk_flush(trk);
      }
      if (INT && t >= 0) { gin += GRID ? N2 : (size_t)SS; gout += GRID ? N2 : (size_t)(PS * PS); }
    }
  }
  flush_counters(c, cx.status);
  flush_speed(best, p.next_speed);
#undef wv
#undef zcur
#undef znxt
}

template <class R, int RECON, int RS, int FAST, int MINB, int GRID, int GC>
__global__ void __launch_bounds__(LEAN_NT, MINB)
ctu_lean_kernel(const R* __restrict__ in, R* __restrict__ out, R* __restrict__ face_flux, int Ng, int g, Par<R> p,
                const R* __restrict__ max_speed, R cfl, long long* status, GridIO<R> gio) {
  constexpr int GW = 2 + RECON, SWP = PS + 2 * GW, WPL = SWP * SWP, NW = 2 * (1 + RECON) + 1;
  constexpr int RC = RECON == RECON_PPM ? 1 : 0, NWS = NW - RC;
  constexpr int NC = LEAN_COLS, NT = LEAN_NT, FT = PS + 2;
  apply_device_dt(p, max_speed, cfl);

  // shared memory: everything at compile-time offsets; the raw planes, whose size depends on g, come last
  extern __shared__ __align__(16) unsigned char smem[];
  LeanCtx<R> cx;
  cx.in = in; cx.out = out; cx.face_flux = face_flux; cx.Ng = Ng; cx.g = g; cx.status = status; cx.gio = gio;
  cx.bar = reinterpret_cast<uint64_t*>(smem);          // [2]
  R* ring = reinterpret_cast<R*>(smem + 64);           // [NWS] fields of WPL cells: primitive planes
  R* zs = ring + NWS * 5 * WPL;                        // [2][2] fields of NT cells: private traced z states (lo, up) of planes t, t+1
  R* xy = zs + 4 * 5 * NT;                             // [6] fields of NC cells: LOX UPX LOY UPY FX FY
  cx.raw = xy + 6 * 5 * NC;                            // [2][5][SS] landing zone of the bulk copies (SoA as in HBM)
#if LEAN_OPAQUE
  // the shared-window address of the tile is formed ONCE and made opaque: ptxas otherwise re-derives it (S2UR SR_CgaCtaId,
  // UMOV, ULEA) at every use inside the loop instead of holding one register
  uint32_t sb = smem_u32(smem);
  asm volatile("" : "+r"(sb));
  cx.sm_bar = sb;
  cx.sm_ring = sb + 64u;
  cx.sm_zs = cx.sm_ring + (uint32_t)(sizeof(R) * NWS * 5 * WPL);
  cx.sm_xy = cx.sm_zs + (uint32_t)(sizeof(R) * 4 * 5 * NT);
  cx.sm_raw = cx.sm_xy + (uint32_t)(sizeof(R) * 6 * 5 * NC);
#else
  cx.sm_bar = smem_u32(smem);
  cx.sm_ring = smem_u32(ring);
  cx.sm_zs = smem_u32(zs);
  cx.sm_xy = smem_u32(xy);
  cx.sm_raw = smem_u32(cx.raw);
#endif

#if LEAN_OPAQUE
  int tid = threadIdx.x;
  asm volatile("" : "+r"(tid));  // one register instead of an S2R at every re-derivation
#else
  const int tid = threadIdx.x;
#endif
  if (tid == 0) {
    mbar_init(cx.bar, 1);
    mbar_init(cx.bar + 1, 1);
    fence_mbar_init();
    fence_async_smem();
  }
  __syncthreads();
  // ---- column and role of this thread
  // warps 0-7: the 256 interior columns (two rows of 16 per warp: no lane idles in the interior-only phases);
  // warp 8: the x ring (i = -1, 16; j = 0..15); warp 9: the y ring (j = -1, 16; i = 0..15)
  int ii, jj;
  if (tid < PS * PS) { jj = 1 + (tid >> 4); ii = 1 + (tid & 15); }
  else if (tid < PS * PS + 32) { const int l = tid - PS * PS; jj = 1 + (l >> 1); ii = (l & 1) ? FT - 1 : 0; }
  else { const int l = tid - PS * FT; jj = (l < PS) ? 0 : FT - 1; ii = 1 + (l & (PS - 1)); }
  if (LEAN_ROLE_SPLIT) {
    if (tid < PS * PS) ctu_lean_role<R, RECON, RS, FAST, GRID, ROLE_INT, GC>(cx, p, ii, jj, tid);
    else if (tid < PS * PS + 32) ctu_lean_role<R, RECON, RS, FAST, GRID, ROLE_XR, GC>(cx, p, ii, jj, tid);
    else ctu_lean_role<R, RECON, RS, FAST, GRID, ROLE_YR, GC>(cx, p, ii, jj, tid);
  } else {
    ctu_lean_role<R, RECON, RS, FAST, GRID, ROLE_ANY, GC>(cx, p, ii, jj, tid);
  }
}

// persistent grid: SMs x resident CTAs per SM (occupancy API), capped at Ng
template <class R, int RECON, int RS, int FAST, int MINB, int GRID = 0, int GC = -1> cudaError_t launch_ctu_lean(const SolveArgs<R>& a) {
  // the default options at the ghost width of the AMR batches (g = 3, BASELINE.json configs[2] and [4]) have their own instantiation
  if constexpr (FAST && !GRID && GC < 0 && (sizeof(R) == 4 || LEAN_GC_F64)) {
    if (a.g == 3) return launch_ctu_lean<R, RECON, RS, FAST, MINB, GRID, 3>(a);
  }
  auto kern = ctu_lean_kernel<R, RECON, RS, FAST, MINB, GRID, GC>;
  const size_t smem = lean_smem_bytes(sizeof(R), RECON, a.g);
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
