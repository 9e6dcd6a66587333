// srpp_probe.cu -- FP32 peak probe: the denominator of "% of FP32 peak" measured on the device the
// solver runs on (MEASURED_PEAKS.json has no FP32 entry, so the harness measures one).
//
// Two register-only FMA streams, 16 independent accumulator chains per thread so that neither the
// 4-cycle FMA latency nor the issue port is the limit:
//   variant 0: scalar FFMA            (2 flop / lane / instruction)
//   variant 1: packed FFMA2 (f32x2)   (4 flop / lane / instruction) -- the form the pair loop uses
// Grid = SMs x resident CTAs, 256 threads, CUDA events on the caller's stream.  The result is what the
// FP32 pipe sustains at the clock the chip holds under THIS kind of load; DESIGN.md compares it with the
// nominal SMs x 128 lanes x 2 flop x f_max.
#include "srpp_internal.cuh"

namespace srpp {

constexpr int kProbeChains = 16;
constexpr int kProbeInner = 64;   // FMA rounds per loop trip (each round = kProbeChains instructions)

__global__ void __launch_bounds__(256) k_probe_ffma(int trips, float a, float b, float* __restrict__ out) {
  float acc[kProbeChains];
#pragma unroll
  for (int k = 0; k < kProbeChains; ++k) acc[k] = (float)(threadIdx.x + k) * 1e-3f;
  for (int t = 0; t < trips; ++t) {
#pragma unroll
    for (int r = 0; r < kProbeInner; ++r) {
#pragma unroll
      for (int k = 0; k < kProbeChains; ++k) acc[k] = __fmaf_rn(acc[k], a, b);
    }
  }
  float s = 0.f;
#pragma unroll
  for (int k = 0; k < kProbeChains; ++k) s += acc[k];
  if (s == 123.456f) out[0] = s;   // keeps the chains alive without a store in the common case
}

__global__ void __launch_bounds__(256) k_probe_ffma2(int trips, float a, float b, float* __restrict__ out) {
  float2 acc[kProbeChains];
  const float2 a2 = make_float2(a, a), b2 = make_float2(b, b);
#pragma unroll
  for (int k = 0; k < kProbeChains; ++k) acc[k] = make_float2((float)(threadIdx.x + k) * 1e-3f, (float)k * 2e-3f);
  for (int t = 0; t < trips; ++t) {
#pragma unroll
    for (int r = 0; r < kProbeInner; ++r) {
#pragma unroll
      for (int k = 0; k < kProbeChains; ++k) acc[k] = __ffma2_rn(acc[k], a2, b2);
    }
  }
  float s = 0.f;
#pragma unroll
  for (int k = 0; k < kProbeChains; ++k) s += acc[k].x + acc[k].y;
  if (s == 123.456f) out[0] = s;
}

// Variants 2 and 3: the same packed stream, but every FFMA2 reads 2 resp. 3 DIFFERENT vector registers (the values
// are thread-dependent so the compiler cannot move them to uniform registers).  On B200 the first sustains the FFMA2
// peak, the second needs 3 pipe cycles per instruction instead of 2: the register file feeds two 64-bit operands per
// instruction slot.  DESIGN.md 5.2 uses this to bound the pair loop (its f and accumulate steps have 3 operands).
template <int kVectorOperands>
__global__ void __launch_bounds__(256) k_probe_ffma2_operands(int trips, float a, float b, float* __restrict__ out) {
  constexpr int kChains = 8;
  unsigned long long d[kChains], A[kChains], B[kChains];
#pragma unroll
  for (int k = 0; k < kChains; ++k) {
    const float t = 1.0f - (float)(threadIdx.x + 1) * 1.0e-9f * (float)(k + 1);   // per-thread, ~1
    float2 dv = make_float2((float)(threadIdx.x + k) * 1e-3f, (float)k * 2e-3f), av = make_float2(a * t, a * t * t), bv = make_float2(b * t, b);
    d[k] = *reinterpret_cast<unsigned long long*>(&dv);
    A[k] = *reinterpret_cast<unsigned long long*>(&av);
    B[k] = *reinterpret_cast<unsigned long long*>(&bv);
  }
  float2 bu = make_float2(b, b);
  const unsigned long long BU = *reinterpret_cast<unsigned long long*>(&bu);
  for (int t = 0; t < trips; ++t) {
#pragma unroll
    for (int r = 0; r < kProbeInner; ++r) {
#pragma unroll
      for (int k = 0; k < kChains; ++k) {
        if (kVectorOperands == 3) asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(d[k]) : "l"(A[k]), "l"(B[k]));
        else asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(d[k]) : "l"(A[k]), "l"(BU));
      }
    }
  }
  float s = 0.f;
#pragma unroll
  for (int k = 0; k < kChains; ++k) { float2 v = *reinterpret_cast<float2*>(&d[k]); s += v.x + v.y; }
  if (s == 123.456f) out[0] = s;
}

cudaError_t run_fp32_probe(cudaStream_t st, int variant, int trips, double* flops_per_s, float* scratch_dev) {
  int dev = 0, sms = 0, occ = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  if (e != cudaSuccess) return e;
  if (variant == 0) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_probe_ffma, 256, 0);
  else if (variant == 1) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_probe_ffma2, 256, 0);
  else if (variant == 2) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_probe_ffma2_operands<2>, 256, 0);
  else e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_probe_ffma2_operands<3>, 256, 0);
  if (e != cudaSuccess) return e;
  if (occ < 1) occ = 1;
  if (occ > 4) occ = 4;
  const int grid = sms * occ;
  cudaEvent_t e0, e1;
  if ((e = cudaEventCreate(&e0)) != cudaSuccess) return e;
  if ((e = cudaEventCreate(&e1)) != cudaSuccess) { cudaEventDestroy(e0); return e; }
  // a = 1 - 2^-20, b = 2^-20: the chains converge to 1 and never overflow, denormalise or get folded away
  const float a = 0.99999905f, b = 9.5367432e-7f;
  for (int rep = 0; rep < 2; ++rep) {   // first launch warms clocks and instruction cache
    cudaEventRecord(e0, st);
    if (variant == 0) k_probe_ffma<<<grid, 256, 0, st>>>(trips, a, b, scratch_dev);
    else if (variant == 1) k_probe_ffma2<<<grid, 256, 0, st>>>(trips, a, b, scratch_dev);
    else if (variant == 2) k_probe_ffma2_operands<2><<<grid, 256, 0, st>>>(trips, a, b, scratch_dev);
    else k_probe_ffma2_operands<3><<<grid, 256, 0, st>>>(trips, a, b, scratch_dev);
    cudaEventRecord(e1, st);
  }
  e = cudaEventSynchronize(e1);
  float ms = 0.f;
  if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  if (e != cudaSuccess) return e;
  const double chains = variant >= 2 ? 8.0 : (double)kProbeChains;
  const double flop = (double)grid * 256.0 * (double)trips * kProbeInner * chains * (variant == 0 ? 2.0 : 4.0);
  *flops_per_s = flop / ((double)ms * 1e-3);
  return cudaGetLastError();
}

}  // namespace srpp
