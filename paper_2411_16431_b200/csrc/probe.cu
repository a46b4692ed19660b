// tn_fp64_peak: measures this GPU's FP64 tensor-core (DMMA) peak, the roofline denominator of every
// dense contraction of the path.  MEASURED_PEAKS.json carries no FP64 figure, so bench.py measures it
// live (profiles/r01_fp64_peak.md records the round-1 sweep over every mma.sync f64 shape).
#include "kernels.cuh"

__global__ void k_dmma_chain(double* out, int iters) {
  double a = 1.0 + threadIdx.x * 1e-9, b = 1.0000001;
  double c[8][2];
#pragma unroll
  for (int j = 0; j < 8; j++) { c[j][0] = j; c[j][1] = j + 0.5; }
  for (int i = 0; i < iters; i++) {
#pragma unroll
    for (int j = 0; j < 8; j++) dmma884(c[j][0], c[j][1], a, b);
  }
  double s = 0;
#pragma unroll
  for (int j = 0; j < 8; j++) s += c[j][0] + c[j][1];
  out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = s;
}

extern "C" int tn_fp64_peak(double* tflops) {
  if (!tflops) return TN_ERR_ARG;
  *tflops = 0.0;
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) {
    cudaGetLastError();
    return TN_ERR_CUDA;
  }
  const int threads = 256, blocks = sms * 8, iters = 4000;
  double* out = nullptr;
  if (cudaMalloc(&out, sizeof(double) * threads * blocks) != cudaSuccess) { cudaGetLastError(); return TN_ERR_OOM; }
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0); cudaEventCreate(&e1);
  k_dmma_chain<<<blocks, threads>>>(out, 100);
  float best = 1e30f;
  for (int r = 0; r < 3; r++) {
    cudaEventRecord(e0);
    k_dmma_chain<<<blocks, threads>>>(out, iters);
    cudaEventRecord(e1);
    cudaEventSynchronize(e1);
    float ms = 0;
    cudaEventElapsedTime(&ms, e0, e1);
    if (ms > 0 && ms < best) best = ms;
  }
  cudaError_t e = cudaDeviceSynchronize();
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  cudaFree(out);
  if (e != cudaSuccess || !(best < 1e29f)) { cudaGetLastError(); return TN_ERR_CUDA; }
  const double flop = 8.0 * (2.0 * 8 * 8 * 4) / 32.0 * (double)iters * threads * blocks;
  *tflops = flop / best * 1e-9;
  return TN_OK;
}
