// hx_probe.cu -- device probe behind hx_probe_fp64(): measures the FP64 FMA issue rate of the
// current GPU (the denominator of the "alu" roofline in DESIGN.md / bench.py) and the latency of a
// dependent DFMA.  Not part of the hydro path; no state, default stream, synchronous.
#include <cuda_runtime.h>

#include "../../include/hx.h"

namespace hx {

// CHAINS independent x <- x*a + b recurrences per thread; a, b arrive as arguments so nothing folds.
template <int CHAINS>
__global__ void __launch_bounds__(256) dfma_chain_kernel(double* out, int iters, double a, double b, long long* cycles) {
  double x[CHAINS];
#pragma unroll
  for (int c = 0; c < CHAINS; ++c) x[c] = 1.0 + 1e-9 * (threadIdx.x + c);
  const long long t0 = clock64();
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int r = 0; r < 8; ++r) {
#pragma unroll
      for (int c = 0; c < CHAINS; ++c) x[c] = fma(x[c], a, b);
    }
  }
  const long long t1 = clock64();
  double s = 0.0;
#pragma unroll
  for (int c = 0; c < CHAINS; ++c) s += x[c];
  if (s == 123.456) out[0] = s;   // keeps the chains alive; never true for the arguments used
  if (cycles && threadIdx.x == 0 && blockIdx.x == 0) cycles[0] = t1 - t0;
}

}  // namespace hx

extern "C" int hx_probe_fp64(double* tflops, double* dep_latency_cycles) {
  using namespace hx;
  if (!tflops || !dep_latency_cycles) return HX_ERR_INVALID_ARG;
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return HX_ERR_CUDA;
  double* d_out = nullptr;
  long long* d_cyc = nullptr;
  if (cudaMalloc(&d_out, sizeof(double)) != cudaSuccess || cudaMalloc(&d_cyc, sizeof(long long)) != cudaSuccess) return HX_ERR_ALLOC;
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0);
  cudaEventCreate(&e1);
  int rc = HX_OK;
  // throughput: 8 CTAs x 256 threads per SM, 8 chains per thread
  const int iters = 2048, chains = 8, grid = sms * 8;
  dfma_chain_kernel<8><<<grid, 256>>>(d_out, 64, 0.999999, 1e-6, nullptr);   // warm-up
  float best = 1e30f;
  for (int rep = 0; rep < 5; ++rep) {
    cudaEventRecord(e0);
    dfma_chain_kernel<8><<<grid, 256>>>(d_out, iters, 0.999999, 1e-6, nullptr);
    cudaEventRecord(e1);
    if (cudaEventSynchronize(e1) != cudaSuccess) { rc = HX_ERR_CUDA; break; }
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    if (ms < best) best = ms;
  }
  if (rc == HX_OK) {
    const double fmas = (double)grid * 256.0 * chains * 8.0 * iters;
    *tflops = 2.0 * fmas / (best * 1e-3) / 1e12;
    // latency: one warp, one chain
    dfma_chain_kernel<1><<<1, 32>>>(d_out, 4096, 0.999999, 1e-6, d_cyc);
    long long cyc = 0;
    if (cudaMemcpy(&cyc, d_cyc, sizeof(cyc), cudaMemcpyDeviceToHost) != cudaSuccess) rc = HX_ERR_CUDA;
    else *dep_latency_cycles = (double)cyc / (4096.0 * 8.0);
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(d_out);
  cudaFree(d_cyc);
  return rc;
}
