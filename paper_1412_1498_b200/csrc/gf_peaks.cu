// gf_peaks.cu — FMA-chain micro-kernel behind gf_peak_fma: the measured FP64 / FP32 CUDA-core peak that the flops leg of
// the roofline divides by ("the builder must measure both with an FMA-chain microbenchmark").
// Not part of the gauge-fixing path: it touches no memory besides one guard word.
#include <cuda_runtime.h>

#include "../../include/gf.h"

namespace {

constexpr int PEAK_THREADS = 256;
constexpr int PEAK_CHAINS = 16;    // independent accumulators per thread: covers the FMA latency at any occupancy
constexpr int PEAK_INNER = 64;     // unrolled FMAs per chain and outer iteration

template <class T>
__global__ void __launch_bounds__(PEAK_THREADS) fma_chain_kernel(int outer, T a, T b, T* __restrict__ sink) {
  T acc[PEAK_CHAINS];
#pragma unroll
  for (int c = 0; c < PEAK_CHAINS; ++c) acc[c] = T(threadIdx.x + c) * T(1e-3);
  for (int o = 0; o < outer; ++o) {
#pragma unroll
    for (int i = 0; i < PEAK_INNER; ++i)
#pragma unroll
      for (int c = 0; c < PEAK_CHAINS; ++c) acc[c] = fma(acc[c], a, b);
  }
  T s = T(0);
#pragma unroll
  for (int c = 0; c < PEAK_CHAINS; ++c) s += acc[c];
  if (s == T(-12345.678)) sink[0] = s;  // never true for the arguments used; keeps the chains alive
}

template <class T>
cudaError_t time_fma(int blocks, int outer, cudaStream_t st, T* sink, float* ms) {
  cudaEvent_t e0, e1;
  cudaError_t e = cudaEventCreate(&e0);
  if (e != cudaSuccess) return e;
  e = cudaEventCreate(&e1);
  if (e != cudaSuccess) { cudaEventDestroy(e0); return e; }
  fma_chain_kernel<T><<<blocks, PEAK_THREADS, 0, st>>>(outer / 8 + 1, T(0.999), T(1e-3), sink);  // warm-up
  cudaEventRecord(e0, st);
  fma_chain_kernel<T><<<blocks, PEAK_THREADS, 0, st>>>(outer, T(0.999), T(1e-3), sink);
  cudaEventRecord(e1, st);
  e = cudaEventSynchronize(e1);
  if (e == cudaSuccess) e = cudaGetLastError();
  if (e == cudaSuccess) e = cudaEventElapsedTime(ms, e0, e1);
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  return e;
}

}  // namespace

extern "C" int gf_peak_fma(int prec, double seconds_target, void* dev_scratch, void* cuda_stream, double* tflops) {
  if (!tflops || !dev_scratch || (prec != GF_FP64 && prec != GF_FP32) || !(seconds_target > 0.0) || seconds_target > 10.0)
    return GF_EINVAL;
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
    return GF_ECUDA;
  const int blocks = sms * 8;  // 2048 threads per SM asked for; the register count lets at least 4 blocks be resident
  cudaStream_t st = (cudaStream_t)cuda_stream;
  // calibrate on a short run, then one run of about seconds_target
  int outer = 256;
  float ms = 0.f;
  double best = 0.0;
  for (int pass = 0; pass < 2; ++pass) {
    cudaError_t e = prec == GF_FP64 ? time_fma<double>(blocks, outer, st, (double*)dev_scratch, &ms)
                                    : time_fma<float>(blocks, outer, st, (float*)dev_scratch, &ms);
    if (e != cudaSuccess || !(ms > 0.f)) return GF_ECUDA;
    const double flops = 2.0 * (double)blocks * PEAK_THREADS * PEAK_CHAINS * PEAK_INNER * (double)outer;
    const double t = flops / (ms * 1e-3) / 1e12;
    best = t > best ? t : best;
    const double scale = seconds_target * 1e3 / ms;
    if (pass == 0) outer = (int)(outer * (scale < 1.0 ? 1.0 : scale > 4096.0 ? 4096.0 : scale));
  }
  *tflops = best;
  return GF_OK;
}
