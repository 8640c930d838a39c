// peaks.cu -- micro-benchmarks behind jenga_measure_peaks (include/jenga.h): the two roofline denominators the
// Jenga step can bind on (SURVEY.md §7 step 0, §8(d) "Peaks (to be measured)"):
//   * FP32 issue rate: dependent-free FFMA streams on every SM (thread-instructions per second, FMA = 1),
//   * shared-memory bandwidth: conflict-free LDS.128 streams on every SM (bytes per second).
// MEASURED_PEAKS.json (driver-written) only has HBM copy bandwidth and bf16 tensor throughput.
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/jenga.h"

namespace jenga_peaks {

constexpr int kThreads = 256, kChains = 8, kInner = 64;

// 8 independent FFMA chains per thread (latency 4, two FMA pipes: 8 chains x 8 warps per scheduler hide it),
// register operands only; the result is written so that nothing is dead code.
__global__ void __launch_bounds__(kThreads) k_ffma(float* out, int outer, float a, float b) {
  float x[kChains];
#pragma unroll
  for (int k = 0; k < kChains; ++k) x[k] = (float)(threadIdx.x + k) * 1.0e-3f;
  for (int it = 0; it < outer; ++it) {
#pragma unroll
    for (int j = 0; j < kInner; ++j)
#pragma unroll
      for (int k = 0; k < kChains; ++k) x[k] = fmaf(x[k], a, b);
  }
  float s = 0.0f;
#pragma unroll
  for (int k = 0; k < kChains; ++k) s += x[k];
  out[(size_t)blockIdx.x * kThreads + threadIdx.x] = s;
}

// The same with three distinct per-thread register operands (no uniform-register or immediate operand): the form
// the solver's FFMAs have.
__global__ void __launch_bounds__(kThreads) k_ffma3(float* out, int outer) {
  float x[kChains];
  const float a = 0.999f + (float)threadIdx.x * 1.0e-7f, b = 1.0e-3f + (float)threadIdx.x * 1.0e-9f;
#pragma unroll
  for (int k = 0; k < kChains; ++k) x[k] = (float)(threadIdx.x + k) * 1.0e-3f;
  for (int it = 0; it < outer; ++it) {
#pragma unroll
    for (int j = 0; j < kInner; ++j)
#pragma unroll
      for (int k = 0; k < kChains; ++k) x[k] = fmaf(x[k], a, b);
  }
  float s = 0.0f;
#pragma unroll
  for (int k = 0; k < kChains; ++k) s += x[k];
  out[(size_t)blockIdx.x * kThreads + threadIdx.x] = s;
}

// FFMAs whose three source registers all change from one instruction to the next (no operand-reuse hits): the shape of
// the solver's cross products and matrix-vector products.  16 accumulators, 8 + 8 multiplicands per thread.
__global__ void __launch_bounds__(kThreads) k_ffma_nr(float* out, int outer) {
  float x[16], y[8], z[8];
#pragma unroll
  for (int k = 0; k < 16; ++k) x[k] = (float)(threadIdx.x + k) * 1.0e-3f;
#pragma unroll
  for (int k = 0; k < 8; ++k) { y[k] = 0.999f + (float)(threadIdx.x + k) * 1.0e-7f; z[k] = 1.0e-3f + (float)(threadIdx.x * 8 + k) * 1.0e-9f; }
  for (int it = 0; it < outer; ++it) {
#pragma unroll
    for (int j = 0; j < kInner / 2; ++j)
#pragma unroll
      for (int k = 0; k < 16; ++k) x[k] = fmaf(y[(k + j) & 7], z[(k + 3 * j + 1) & 7], x[k]);
  }
  float s = 0.0f;
#pragma unroll
  for (int k = 0; k < 16; ++k) s += x[k];
  out[(size_t)blockIdx.x * kThreads + threadIdx.x] = s;
}

// The packed form of sm_100 (fma.rn.f32x2, SASS FFMA2): two FMAs per thread per instruction on 64-bit register pairs, again
// with no operand reuse.  Counted as two FP32 thread-instructions each.
__global__ void __launch_bounds__(kThreads) k_ffma2_nr(float* out, int outer) {
  float2 x[8], y[4], z[4];
#pragma unroll
  for (int k = 0; k < 8; ++k) x[k] = make_float2((float)(threadIdx.x + k) * 1.0e-3f, (float)(threadIdx.x + k) * 2.0e-3f);
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    y[k] = make_float2(0.999f + (float)(threadIdx.x + k) * 1.0e-7f, 0.998f + (float)(threadIdx.x + k) * 1.0e-7f);
    z[k] = make_float2(1.0e-3f + (float)(threadIdx.x * 8 + k) * 1.0e-9f, 2.0e-3f + (float)(threadIdx.x * 8 + k) * 1.0e-9f);
  }
  for (int it = 0; it < outer; ++it) {
#pragma unroll
    for (int j = 0; j < kInner / 2; ++j)
#pragma unroll
      for (int k = 0; k < 8; ++k) x[k] = __ffma2_rn(y[(k + j) & 3], z[(k + 3 * j + 1) & 3], x[k]);
  }
  float s = 0.0f;
#pragma unroll
  for (int k = 0; k < 8; ++k) s += x[k].x + x[k].y;
  out[(size_t)blockIdx.x * kThreads + threadIdx.x] = s;
}

// Every lane reads consecutive 16-byte words (conflict-free LDS.128, 4 wavefronts of 128 B per instruction);
// 8 loads in flight per thread per inner step; the sums keep the loads alive.
__global__ void __launch_bounds__(kThreads) k_lds(float* out, int outer) {
  extern __shared__ float4 sm4[];
  const int n4 = 8 * kThreads;                               // 32 KB per CTA
  for (int i = threadIdx.x; i < n4; i += kThreads) sm4[i] = make_float4((float)i, 1.0f, 2.0f, 3.0f);
  __syncthreads();
  float4 acc = make_float4(0, 0, 0, 0);
  int base = threadIdx.x;
  for (int it = 0; it < outer; ++it) {
#pragma unroll
    for (int j = 0; j < 8; ++j) {
      const float4 v = sm4[(base + j * kThreads) & (n4 - 1)];
      acc.x += v.x; acc.y += v.y; acc.z += v.z; acc.w += v.w;
    }
    base = (base + 32) & (n4 - 1);
  }
  out[(size_t)blockIdx.x * kThreads + threadIdx.x] = acc.x + acc.y + acc.z + acc.w;
}

}  // namespace jenga_peaks

// out[0] = FP32 thread-instructions per second (FFMA, all SMs), out[1] = shared-memory bytes per second (LDS.128),
// out[2] = SM count, out[3] = seconds of the FFMA run, out[4] = seconds of the LDS run, out[5] = FP32 thread-instructions
// per second of the three-register-operand FFMA form, out[6] = the same with three source registers that all change from
// one instruction to the next (no operand-reuse hits).
// `scratch` is a caller-owned device buffer of at least jenga_peaks_scratch_bytes(); the call synchronises the
// stream (it is a measurement, not a step of the path).
extern "C" size_t jenga_peaks_scratch_bytes(void) { return (size_t)148 * 8 * 8 * jenga_peaks::kThreads * sizeof(float); }

extern "C" int jenga_measure_peaks(double* out, void* scratch, void* cuda_stream) {
  using namespace jenga_peaks;
  if (!out || !scratch) return JENGA_E_ARG;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  int dev = 0, n_sm = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return JENGA_E_CUDA;
  cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0); cudaEventCreate(&e1);
  float* o = (float*)scratch;
  const int grid = n_sm * 8;                                  // 8 CTAs of 256 threads per SM = 64 warps per SM
  const int outer_f = 4096, outer_l = 2048;
  float ms_f = 1e30f, ms_l = 1e30f;
  cudaFuncSetAttribute(k_lds, cudaFuncAttributeMaxDynamicSharedMemorySize, 8 * kThreads * 16);
  for (int rep = 0; rep < 4; ++rep) {                         // first rep warms up; best of the rest
    cudaEventRecord(e0, st);
    k_ffma<<<grid, kThreads, 0, st>>>(o, outer_f, 0.999f, 1.0e-3f);
    cudaEventRecord(e1, st);
    if (cudaEventSynchronize(e1) != cudaSuccess) return JENGA_E_CUDA;
    float ms; cudaEventElapsedTime(&ms, e0, e1);
    if (rep && ms < ms_f) ms_f = ms;
  }
  float ms_f3 = 1e30f;
  for (int rep = 0; rep < 4; ++rep) {
    cudaEventRecord(e0, st);
    k_ffma3<<<grid, kThreads, 0, st>>>(o, outer_f);
    cudaEventRecord(e1, st);
    if (cudaEventSynchronize(e1) != cudaSuccess) return JENGA_E_CUDA;
    float ms; cudaEventElapsedTime(&ms, e0, e1);
    if (rep && ms < ms_f3) ms_f3 = ms;
  }
  float ms_nr = 1e30f;
  for (int rep = 0; rep < 4; ++rep) {
    cudaEventRecord(e0, st);
    k_ffma_nr<<<grid, kThreads, 0, st>>>(o, outer_f);
    cudaEventRecord(e1, st);
    if (cudaEventSynchronize(e1) != cudaSuccess) return JENGA_E_CUDA;
    float ms; cudaEventElapsedTime(&ms, e0, e1);
    if (rep && ms < ms_nr) ms_nr = ms;
  }
  float ms_p2 = 1e30f;
  for (int rep = 0; rep < 4; ++rep) {
    cudaEventRecord(e0, st);
    k_ffma2_nr<<<grid, kThreads, 0, st>>>(o, outer_f);
    cudaEventRecord(e1, st);
    if (cudaEventSynchronize(e1) != cudaSuccess) return JENGA_E_CUDA;
    float ms; cudaEventElapsedTime(&ms, e0, e1);
    if (rep && ms < ms_p2) ms_p2 = ms;
  }
  const int grid_l = n_sm * 6;                                // 6 x 32 KB of shared memory per SM
  for (int rep = 0; rep < 4; ++rep) {
    cudaEventRecord(e0, st);
    k_lds<<<grid_l, kThreads, 8 * kThreads * 16, st>>>(o, outer_l);
    cudaEventRecord(e1, st);
    if (cudaEventSynchronize(e1) != cudaSuccess) return JENGA_E_CUDA;
    float ms; cudaEventElapsedTime(&ms, e0, e1);
    if (rep && ms < ms_l) ms_l = ms;
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  if (cudaGetLastError() != cudaSuccess) return JENGA_E_CUDA;
  const double n_ffma = (double)grid * kThreads * (double)outer_f * kInner * kChains;
  const double n_bytes = (double)grid_l * kThreads * (double)outer_l * 8 * 16;
  out[0] = n_ffma / (ms_f * 1e-3); out[1] = n_bytes / (ms_l * 1e-3); out[2] = (double)n_sm;
  out[3] = ms_f * 1e-3; out[4] = ms_l * 1e-3; out[5] = n_ffma / (ms_f3 * 1e-3);
  out[6] = n_ffma / (ms_nr * 1e-3);
  out[7] = n_ffma / (ms_p2 * 1e-3);
  return JENGA_OK;
}
