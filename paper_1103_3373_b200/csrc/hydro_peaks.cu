// hydro_peaks.cu -- register-resident ALU loops that MEASURE the roofline denominators of the ALU-bound kernels
// ("FP32 and FP64 FMA peaks must be measured on the box with a register-resident FFMA / DFMA loop at
// the clocks the kernel actually sustains").  bench.py --table peaks times them with CUDA events under the clock
// sampler and writes profiles/alu_peaks.json; bench.py reads that file for `roofline.peak`.
//
// Every thread carries CH independent accumulator chains (so that neither the 4-cycle FMA latency nor the issue
// port limits the loop) and runs `iters` passes of UNROLL x CH operations; operands never leave registers.
// Measurement helper, not part of the update path.
#include <cuda_runtime.h>
#include <cstdint>

#include "../../include/hydro.h"

namespace hydro {

constexpr int PEAK_CH = 16, PEAK_UNROLL = 8;

__device__ __forceinline__ uint64_t pk2(float a, float b) { uint64_t r; asm("mov.b64 %0, {%1,%2};" : "=l"(r) : "f"(a), "f"(b)); return r; }
__device__ __forceinline__ void upk2(uint64_t v, float& a, float& b) { asm("mov.b64 {%0,%1}, %2;" : "=f"(a), "=f"(b) : "l"(v)); }
__device__ __forceinline__ uint64_t fma2(uint64_t a, uint64_t b, uint64_t c) {
  uint64_t r;
  asm volatile("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
  return r;
}

// kind 0: FFMA   kind 3: FMUL / FADD alternating   kind 4: FFMA : FMNMX 1:1 (do the FMA and ALU pipes issue side by side?)
// kind 7: FFMA with both multiplicand and addend taken from the constant bank (kernel parameters) instead of registers
template <int KIND> __global__ void __launch_bounds__(512) peak_f32(float* out, float a0, float b0, int iters) {
  float acc[PEAK_CH], alt[PEAK_CH];
  // register operands (the form a real kernel issues): made thread-dependent so that they cannot live in the constant bank
  const float a = KIND == 7 ? a0 : a0 + 1e-9f * (float)threadIdx.x, b = KIND == 7 ? b0 : b0 + 1e-12f * (float)threadIdx.x;
#pragma unroll
  for (int c = 0; c < PEAK_CH; ++c) { acc[c] = a * (float)(threadIdx.x + c); alt[c] = b + (float)c; }
#pragma unroll 1
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int u = 0; u < PEAK_UNROLL; ++u) {
#pragma unroll
      for (int c = 0; c < PEAK_CH; ++c) {
        if (KIND == 0 || KIND == 7) acc[c] = fmaf(acc[c], a, b);
        if (KIND == 3) acc[c] = (u & 1) ? __fmul_rn(acc[c], a) : __fadd_rn(acc[c], b);
        if (KIND == 4) { acc[c] = fmaf(acc[c], a, b); alt[c] = fminf(alt[c], acc[(c + 5) % PEAK_CH]); }
      }
    }
  }
  float s = 0.f;
#pragma unroll
  for (int c = 0; c < PEAK_CH; ++c) s += acc[c] + (KIND == 4 ? alt[c] : 0.f);
  if (s == 123.456f) out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

// kind 1: FFMA2 (fma.rn.f32x2, two FMAs per instruction)   kind 5: FFMA2 : FMNMX 1:1
template <int KIND> __global__ void __launch_bounds__(512) peak_f32x2(float* out, float a, float b, int iters) {
  uint64_t acc[PEAK_CH];
  float alt[PEAK_CH];
  const float ta = 1e-9f * (float)threadIdx.x;
  const uint64_t A = pk2(a + ta, a + 1e-3f), B = pk2(b - ta, b - 1e-3f);
#pragma unroll
  for (int c = 0; c < PEAK_CH; ++c) { acc[c] = pk2(a * (float)(threadIdx.x + c), b * (float)c); alt[c] = b + (float)c; }
#pragma unroll 1
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int u = 0; u < PEAK_UNROLL; ++u) {
#pragma unroll
      for (int c = 0; c < PEAK_CH; ++c) {
        acc[c] = fma2(acc[c], A, B);
        if (KIND == 5) { float x, y; upk2(acc[(c + 5) % PEAK_CH], x, y); alt[c] = fminf(alt[c], x); }
      }
    }
  }
  float s = 0.f;
#pragma unroll
  for (int c = 0; c < PEAK_CH; ++c) { float x, y; upk2(acc[c], x, y); s += x + y + (KIND == 5 ? alt[c] : 0.f); }
  if (s == 123.456f) out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

// kind 2: DFMA
__global__ void __launch_bounds__(512) peak_f64(double* out, double a, double b, int iters) {
  double acc[PEAK_CH];
#pragma unroll
  for (int c = 0; c < PEAK_CH; ++c) acc[c] = a * (double)(threadIdx.x + c);
#pragma unroll 1
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int u = 0; u < PEAK_UNROLL; ++u) {
#pragma unroll
      for (int c = 0; c < PEAK_CH; ++c) acc[c] = fma(acc[c], a, b);
    }
  }
  double s = 0.0;
#pragma unroll
  for (int c = 0; c < PEAK_CH; ++c) s += acc[c];
  if (s == 123.456) out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

// kind 6: MUFU (rsqrt.approx.ftz.f32; ptxas folds pairs of rcp.approx away), the unit behind the fp32 divisions / square roots
__global__ void __launch_bounds__(512) peak_mufu(float* out, float a, int iters) {
  float acc[PEAK_CH];
#pragma unroll
  for (int c = 0; c < PEAK_CH; ++c) acc[c] = a + (float)(threadIdx.x + c);
#pragma unroll 1
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int u = 0; u < PEAK_UNROLL; ++u) {
#pragma unroll
      for (int c = 0; c < PEAK_CH; ++c) { float r; asm volatile("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(acc[c])); acc[c] = r; }
    }
  }
  float s = 0.f;
#pragma unroll
  for (int c = 0; c < PEAK_CH; ++c) s += acc[c];
  if (s == 123.456f) out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

// kinds 8-13: does the packed FFMA2 relieve the ISSUE port?  Equal arithmetic as 2 x FFMA or 1 x FFMA2 per unit, mixed with the
// other instruction classes of the hydro kernels (NA x (FSETP + FSEL), NM x MUFU.RSQ, NI x SHF, all on independent chains).
// Measured on B200 (profiles/alu_peaks.json "issue_probe"): the packed form is never faster -- FFMA2 holds the issue port like
// two FFMAs -- which is why the fused kernels do not use it.
__device__ __forceinline__ float fma1(float a, float b, float c) { float r; asm volatile("fma.rn.f32 %0, %1, %2, %3;" : "=f"(r) : "f"(a), "f"(b), "f"(c)); return r; }
template <int PACKED, int NF, int NA, int NM, int NI>
__global__ void __launch_bounds__(512) issue_probe(float* out, float a0, float b0, int iters) {
  constexpr int CH = 8;
  const float t = 1e-9f * threadIdx.x;
  const float a = a0 + t, b = b0 - t;
  int sh = threadIdx.x & 7;
  const uint64_t A = pk2(a, a + 1e-3f), B = pk2(b, b - 1e-3f);
  float acc[CH * 2], alt[CH], mu[CH];
  uint64_t acc2[CH];
  int ia[CH];
#pragma unroll
  for (int c = 0; c < CH; ++c) {
    acc[2 * c] = a * (threadIdx.x + c); acc[2 * c + 1] = b * c; acc2[c] = pk2(acc[2 * c], acc[2 * c + 1]);
    alt[c] = b + c; ia[c] = threadIdx.x + c; mu[c] = 1.5f + c;
  }
#pragma unroll 1
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int u = 0; u < 4; ++u) {
#pragma unroll
      for (int c = 0; c < CH; ++c) {
#pragma unroll
        for (int f = 0; f < NF; ++f) {
          if (PACKED) acc2[c] = fma2(acc2[c], A, B);
          else { acc[2 * c] = fma1(acc[2 * c], a, b); acc[2 * c + 1] = fma1(acc[2 * c + 1], a, b); }
        }
#pragma unroll
        for (int f = 0; f < NA; ++f) {
          const float o = alt[(c + 1 + f) % CH];
          asm volatile("{.reg .pred p; setp.gt.f32 p, %0, %1; selp.f32 %0, %1, %2, p;}" : "+f"(alt[c]) : "f"(o), "f"(b));
        }
#pragma unroll
        for (int f = 0; f < NM; ++f) { float r; asm volatile("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(mu[c])); mu[c] = r; }
#pragma unroll
        for (int f = 0; f < NI; ++f) asm volatile("shf.l.wrap.b32 %0, %0, %0, %1;" : "+r"(ia[c]) : "r"(sh));
      }
    }
  }
  float s = 0.f;
#pragma unroll
  for (int c = 0; c < CH; ++c) { float x, y; upk2(acc2[c], x, y); s += x + y + acc[2 * c] + acc[2 * c + 1] + alt[c] + mu[c] + (float)ia[c]; }
  if (s == 123.456f) out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

}  // namespace hydro

extern "C" int hydro_alu_peak_launch(int kind, int blocks, int threads, int iters, void* scratch, double* ops_per_launch,
                                     hydro_stream_t stream) {
  using namespace hydro;
  if (kind < 0 || kind > 13) return HYDRO_E_ENUM;
  if (blocks < 1 || threads < 32 || threads > 512 || (threads & 31) || iters < 1) return HYDRO_E_VALUE;
  if (!scratch) return HYDRO_E_NULL;
  cudaStream_t st = (cudaStream_t)stream;
  const double inst = (double)blocks * threads * iters * PEAK_UNROLL * PEAK_CH;  // thread-level operations of the timed kind
  double per = 2.0;
  switch (kind) {
    case 0: peak_f32<0><<<blocks, threads, 0, st>>>((float*)scratch, 1.0000001f, 1e-9f, iters); break;
    case 1: peak_f32x2<1><<<blocks, threads, 0, st>>>((float*)scratch, 1.0000001f, 1e-9f, iters); per = 4.0; break;
    case 2: peak_f64<<<blocks, threads, 0, st>>>((double*)scratch, 1.0000001, 1e-9, iters); break;
    case 3: peak_f32<3><<<blocks, threads, 0, st>>>((float*)scratch, 1.0000001f, 1e-9f, iters); per = 1.0; break;
    case 4: peak_f32<4><<<blocks, threads, 0, st>>>((float*)scratch, 1.0000001f, 1e-9f, iters); break;          // flops of the FFMAs only
    case 5: peak_f32x2<5><<<blocks, threads, 0, st>>>((float*)scratch, 1.0000001f, 1e-9f, iters); per = 4.0; break;
    case 7: peak_f32<7><<<blocks, threads, 0, st>>>((float*)scratch, 1.0000001f, 1e-9f, iters); break;
    // issue probes: ops_per_launch = the FP32 flops of the unit (4 per FFMA pair / FFMA2); 8 chains x 4 unrolls per iteration
    case 8: issue_probe<0, 1, 0, 0, 1><<<blocks, threads, 0, st>>>((float*)scratch, 1.0000001f, 1e-9f, iters); per = 1.0; break;   // 2 FFMA + SHF
    case 9: issue_probe<1, 1, 0, 0, 1><<<blocks, threads, 0, st>>>((float*)scratch, 1.0000001f, 1e-9f, iters); per = 1.0; break;   // FFMA2 + SHF
    case 10: issue_probe<0, 3, 1, 0, 1><<<blocks, threads, 0, st>>>((float*)scratch, 1.0000001f, 1e-9f, iters); per = 3.0; break;  // 6 FFMA + FSETP/FSEL + SHF
    case 11: issue_probe<1, 3, 1, 0, 1><<<blocks, threads, 0, st>>>((float*)scratch, 1.0000001f, 1e-9f, iters); per = 3.0; break;  // 3 FFMA2 + ...
    case 12: issue_probe<0, 4, 1, 1, 1><<<blocks, threads, 0, st>>>((float*)scratch, 1.0000001f, 1e-9f, iters); per = 4.0; break;  // 8 FFMA + FSETP/FSEL + MUFU + SHF
    case 13: issue_probe<1, 4, 1, 1, 1><<<blocks, threads, 0, st>>>((float*)scratch, 1.0000001f, 1e-9f, iters); per = 4.0; break;  // 4 FFMA2 + ...
    default: peak_mufu<<<blocks, threads, 0, st>>>((float*)scratch, 1.5f, iters); per = 1.0; break;
  }
  if (kind >= 8) {  // issue probes: 8 chains x 4 unrolls per pass instead of 16 x 8; `per` = FFMA pairs per unit, 4 flops each
    if (ops_per_launch) *ops_per_launch = (double)blocks * threads * iters * 4 * 8 * per * 4.0;
    return (int)cudaGetLastError();
  }
  if (ops_per_launch) *ops_per_launch = inst * per;
  return (int)cudaGetLastError();
}
