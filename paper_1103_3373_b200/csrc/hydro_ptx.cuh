// hydro_ptx.cuh -- PTX helpers shared by the fused kernels: mbarrier, 1-D bulk async copy (the TMA
// engine without a tensor map), named barriers, strided 5-vector loads / stores.
#pragma once
#include <cstdint>
#include "hydro_math.cuh"

namespace hydro {

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint64_t* bar, uint32_t parity) {
  uint32_t ok;
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
      "selp.u32 %0, 1, 0, p;\n\t}"
      : "=r"(ok)
      : "r"(smem_u32(bar)), "r"(parity)
      : "memory");
  return ok != 0;
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  while (!mbar_try_wait(bar, parity)) {}
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)),
               "l"(src), "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}
__device__ __forceinline__ void fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void fence_mbar_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
// element-wise asynchronous copies global -> shared (LDGSTS): no registers held while the data is in flight
__device__ __forceinline__ void cp_async_elem(float* dst, const float* src) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(smem_u32(dst)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_elem(double* dst, const double* src) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(smem_u32(dst)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }
template <int ID, int N> __device__ __forceinline__ void group_bar() {
  asm volatile("bar.sync %0, %1;" ::"n"(ID), "n"(N) : "memory");
}

template <class R> __device__ __forceinline__ V5<R> ld5(const R* p, int stride) {
  V5<R> x;
#pragma unroll
  for (int q = 0; q < 5; ++q) x[q] = p[q * stride];
  return x;
}
template <class R> __device__ __forceinline__ void st5(R* p, int stride, const V5<R>& x) {
#pragma unroll
  for (int q = 0; q < 5; ++q) p[q * stride] = x[q];
}


// Packed 5-vector fields in shared memory ("4+1" layout): a field of N cells is [N] 16-byte vectors holding
// components 0..3 followed by [N] scalars holding component 4 (float), or [N] (q0,q1) | [N] (q2,q3) | [N] q4
// (double), so that a state moves with 2 (3) shared-memory instructions instead of 5.  N even, base 16-byte aligned.
__device__ __forceinline__ V5<float> ldv(const float* f, int N, int i) {
  const float4 a = reinterpret_cast<const float4*>(f)[i];
  V5<float> x;
  x[0] = a.x; x[1] = a.y; x[2] = a.z; x[3] = a.w; x[4] = f[4 * N + i];
  return x;
}
__device__ __forceinline__ void stv(float* f, int N, int i, const V5<float>& x) {
  reinterpret_cast<float4*>(f)[i] = make_float4(x[0], x[1], x[2], x[3]);
  f[4 * N + i] = x[4];
}
__device__ __forceinline__ V5<double> ldv(const double* f, int N, int i) {
  const double2 a = reinterpret_cast<const double2*>(f)[i], b = reinterpret_cast<const double2*>(f + 2 * N)[i];
  V5<double> x;
  x[0] = a.x; x[1] = a.y; x[2] = b.x; x[3] = b.y; x[4] = f[4 * N + i];
  return x;
}
__device__ __forceinline__ void stv(double* f, int N, int i, const V5<double>& x) {
  reinterpret_cast<double2*>(f)[i] = make_double2(x[0], x[1]);
  reinterpret_cast<double2*>(f + 2 * N)[i] = make_double2(x[2], x[3]);
  f[4 * N + i] = x[4];
}


// The same packed fields addressed by 32-bit shared-space byte addresses, so that every access of the fused kernels is
// `LDS/STS [R + immediate]` off a per-thread address register formed once per kernel (no per-access index arithmetic):
// v = address of the thread's 16-byte vector part, s = address of its scalar part; N = cells per field (compile time).
// A neighbour k cells away is (v + 16 k, s + k sizeof(R)); the scalar part of cell i sits at s = v + Fld::SD - (16 - sizeof(R)) i.
template <class R, int N> struct Fld;
// plain C++ accesses through shared-window pointers rebuilt from the 32-bit addresses: the compiler keeps its freedom to
// hoist and batch the loads of a phase (inline-asm accesses serialised them: 3.0 -> 3.9 ms) and still emits LDS/STS [R + imm]
template <class T> __device__ __forceinline__ T* sm_ptr(uint32_t a) { return static_cast<T*>(__cvta_shared_to_generic((size_t)a)); }
template <int N> struct Fld<float, N> {
  static constexpr uint32_t SD = 16u * N;  // scalar part of cell 0 relative to its vector part
  static constexpr uint32_t BYTES = 20u * N;
  static __device__ __forceinline__ V5<float> ld(uint32_t v, uint32_t s) {
    const float4 a = *sm_ptr<const float4>(v);
    V5<float> x;
    x[0] = a.x; x[1] = a.y; x[2] = a.z; x[3] = a.w; x[4] = *sm_ptr<const float>(s);
    return x;
  }
  static __device__ __forceinline__ void st(uint32_t v, uint32_t s, const V5<float>& x) {
    *sm_ptr<float4>(v) = make_float4(x[0], x[1], x[2], x[3]);
    *sm_ptr<float>(s) = x[4];
  }
};
template <int N> struct Fld<double, N> {
  static constexpr uint32_t SD = 32u * N;
  static constexpr uint32_t BYTES = 40u * N;
  static __device__ __forceinline__ V5<double> ld(uint32_t v, uint32_t s) {
    const double2 a = *sm_ptr<const double2>(v), b = *sm_ptr<const double2>(v + 16u * N);
    V5<double> x;
    x[0] = a.x; x[1] = a.y; x[2] = b.x; x[3] = b.y; x[4] = *sm_ptr<const double>(s);
    return x;
  }
  static __device__ __forceinline__ void st(uint32_t v, uint32_t s, const V5<double>& x) {
    *sm_ptr<double2>(v) = make_double2(x[0], x[1]);
    *sm_ptr<double2>(v + 16u * N) = make_double2(x[2], x[3]);
    *sm_ptr<double>(s) = x[4];
  }
};

}  // namespace hydro
