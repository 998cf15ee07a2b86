// fp64 roof probe: the deposition is bound by the fp64 pipe, and
// MEASURED_PEAKS.json has no fp64 entry, so the harness measures the DFMA rate of the device it
// runs on.  8 independent FMA chains per thread, 4 x 512 threads per SM, CUDA events around one
// launch after a warm-up launch.  Not part of the hot path.
#include "orb_internal.h"

namespace orb {

__global__ void __launch_bounds__(512) k_probe_dfma(double* out, int iters) {
  double a0 = threadIdx.x * 1e-3, a1 = a0 + 1, a2 = a0 + 2, a3 = a0 + 3, a4 = a0 + 4, a5 = a0 + 5,
         a6 = a0 + 6, a7 = a0 + 7;
  const double m = 1.0000001, c = 1e-9;
  for (int i = 0; i < iters; ++i) {
    a0 = fma(a0, m, c); a1 = fma(a1, m, c); a2 = fma(a2, m, c); a3 = fma(a3, m, c);
    a4 = fma(a4, m, c); a5 = fma(a5, m, c); a6 = fma(a6, m, c); a7 = fma(a7, m, c);
  }
  out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = a0 + a1 + a2 + a3 + a4 + a5 + a6 + a7;
}

}  // namespace orb

extern "C" int orb_probe_dfma(int32_t device, double* tflops) {
  if (!tflops) return ORB_E_INVAL;
  int prev = -1, ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) {
    cudaGetLastError();
    return ORB_E_CUDA;
  }
  cudaGetDevice(&prev);
  if (cudaSetDevice(device) != cudaSuccess) return ORB_E_CUDA;
  int sms = 0;
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device);
  const int blocks = sms * 4, threads = 512, iters = 1 << 15;
  double* out = nullptr;
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  int rc = ORB_E_CUDA;
  float ms = 0.f;
  if (cudaMalloc(&out, (size_t)blocks * threads * sizeof(double)) == cudaSuccess &&
      cudaEventCreate(&e0) == cudaSuccess && cudaEventCreate(&e1) == cudaSuccess) {
    orb::k_probe_dfma<<<blocks, threads>>>(out, iters);   // warm-up
    cudaEventRecord(e0);
    orb::k_probe_dfma<<<blocks, threads>>>(out, iters);
    cudaEventRecord(e1);
    if (cudaEventSynchronize(e1) == cudaSuccess && cudaEventElapsedTime(&ms, e0, e1) == cudaSuccess &&
        ms > 0.f) {
      const double fma_count = (double)blocks * threads * 8.0 * iters;
      *tflops = 2.0 * fma_count / (ms * 1e-3) / 1e12;
      rc = ORB_OK;
    }
  }
  cudaGetLastError();
  if (e0) cudaEventDestroy(e0);
  if (e1) cudaEventDestroy(e1);
  cudaFree(out);
  if (prev >= 0) cudaSetDevice(prev);
  return rc;
}
