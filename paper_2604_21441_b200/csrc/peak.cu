// peak.cu -- the measured FP32-pipe peak the AEV kernels' roofline fractions are quoted against (BASELINE.md section 4:
// "a register-resident FMA loop ... before any roofline fraction is quoted").  MEASURED_PEAKS.json
// holds the HBM and tensor peaks only, so bench.py calls nnp_debug_fp32_peak once per run and reports the number beside
// every "alu" fraction.  Two register-resident loops, each thread holding 16 independent accumulator chains:
//   variant 0: scalar FFMA with three register operands (the instruction the AEV kernels are made of);
//   variant 1: packed FFMA2 (fma.rn.f32x2, new on sm_100: two FMAs per issue slot).
// 2 flop per FMA lane.  Grid = 8 blocks of 256 threads per SM, timed with CUDA events on the given stream, best of 5.
#include <algorithm>
#include "nnp_internal.h"

namespace nnp {

constexpr int PEAK_CHAINS = 16;
constexpr int PEAK_ITERS = 2048;

__global__ void __launch_bounds__(256) k_peak_ffma(float* __restrict__ out, float a, float b, int iters) {
  float x[PEAK_CHAINS];
#pragma unroll
  for (int i = 0; i < PEAK_CHAINS; ++i) x[i] = (float)(threadIdx.x + i);
  // a and b live in registers (kernel parameters copied): the 3-register form, not the immediate form
  float ra = a, rb = b;
  asm volatile("" : "+f"(ra), "+f"(rb));
#pragma unroll 1
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int i = 0; i < PEAK_CHAINS; ++i) x[i] = fmaf(x[i], ra, rb);
  }
  float s = 0.f;
#pragma unroll
  for (int i = 0; i < PEAK_CHAINS; ++i) s += x[i];
  if (s == 123.456f) out[blockIdx.x * blockDim.x + threadIdx.x] = s;   // never true: keeps the chains alive
}

__global__ void __launch_bounds__(256) k_peak_ffma2(float* __restrict__ out, float a, float b, int iters) {
  float2 x[PEAK_CHAINS / 2];
#pragma unroll
  for (int i = 0; i < PEAK_CHAINS / 2; ++i) x[i] = make_float2((float)(threadIdx.x + i), (float)(threadIdx.x - i));
  float2 ra = make_float2(a, a * 0.5f), rb = make_float2(b, b * 0.25f);
  asm volatile("" : "+f"(ra.x), "+f"(ra.y), "+f"(rb.x), "+f"(rb.y));
#pragma unroll 1
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int r = 0; r < 2; ++r)
#pragma unroll
      for (int i = 0; i < PEAK_CHAINS / 2; ++i) x[i] = __ffma2_rn(x[i], ra, rb);
  }
  float s = 0.f;
#pragma unroll
  for (int i = 0; i < PEAK_CHAINS / 2; ++i) s += x[i].x + x[i].y;
  if (s == 123.456f) out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

}  // namespace nnp

extern "C" int nnp_debug_fp32_peak(void* cuda_stream, int32_t variant, double* h_tflops) {
  using namespace nnp;
  if (!h_tflops || (variant != 0 && variant != 1)) return NNP_ERR_INVALID_ARG;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms < 1) {
    cudaGetLastError();
    return NNP_ERR_CUDA;
  }
  const int blocks = sms * 8, threads = 256;
  float* d_out = nullptr;
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  if (cudaMalloc(&d_out, sizeof(float) * (size_t)blocks * threads) != cudaSuccess || cudaEventCreate(&e0) != cudaSuccess ||
      cudaEventCreate(&e1) != cudaSuccess) {
    cudaGetLastError();
    if (d_out) cudaFree(d_out);
    if (e0) cudaEventDestroy(e0);
    return NNP_ERR_CUDA;
  }
  double best = 0.0;
  for (int rep = 0; rep < 6; ++rep) {   // rep 0 warms up
    cudaEventRecord(e0, st);
    if (variant == 0) k_peak_ffma<<<blocks, threads, 0, st>>>(d_out, 0.999f, 1.0e-3f, PEAK_ITERS);
    else k_peak_ffma2<<<blocks, threads, 0, st>>>(d_out, 0.999f, 1.0e-3f, PEAK_ITERS);
    cudaEventRecord(e1, st);
    if (cudaEventSynchronize(e1) != cudaSuccess) break;
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    // per iteration and thread: variant 0 = PEAK_CHAINS FMAs; variant 1 = two rounds of PEAK_CHAINS / 2 packed
    // instructions of two FMA lanes each = 2 * PEAK_CHAINS FMAs
    const double fmas = (variant == 0 ? 1.0 : 2.0) * PEAK_CHAINS;
    const double flop = 2.0 * fmas * (double)PEAK_ITERS * (double)blocks * threads;
    if (rep > 0 && ms > 0.f) best = std::max(best, flop / (ms * 1e-3) / 1e12);
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(d_out);
  if (cudaGetLastError() != cudaSuccess || best <= 0.0) return NNP_ERR_CUDA;
  *h_tflops = best;
  return NNP_OK;
}
