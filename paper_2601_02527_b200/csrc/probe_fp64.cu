// probe_fp64.cu -- measurement tool of bench.py, NOT part of the product library (libsmolgp_b200.so):
// a register-only FP64 FMA loop that measures the plain-ALU FP64 throughput of the device the bench runs
// on (the roofline denominator; MEASURED_PEAKS.json has no FP64 entry).  Built by _build.py as its own
// shared object, libsmolgp_probe.so.
#include <cuda_runtime.h>

__global__ void __launch_bounds__(256) k_probe_dfma(double* out, int iters) {
  double a0 = threadIdx.x * 1e-3, a1 = a0 + 1, a2 = a0 + 2, a3 = a0 + 3, a4 = a0 + 4, a5 = a0 + 5, a6 = a0 + 6, a7 = a0 + 7;
  const double m = 0.999999, c = 1e-9;
  for (int i = 0; i < iters; ++i) {
    a0 = fma(a0, m, c); a1 = fma(a1, m, c); a2 = fma(a2, m, c); a3 = fma(a3, m, c);
    a4 = fma(a4, m, c); a5 = fma(a5, m, c); a6 = fma(a6, m, c); a7 = fma(a7, m, c);
  }
  const double s = a0 + a1 + a2 + a3 + a4 + a5 + a6 + a7;
  if (s == 123.456) out[0] = s;
}

// best of `reps` timed launches on the current device's default stream; returns 0 or a cudaError_t
extern "C" int sgprobe_fp64(int device, int reps, double* tflops) {
  if (!tflops) return -1;
  cudaError_t e = cudaSetDevice(device);
  if (e != cudaSuccess) return (int)e;
  int sms = 0;
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device);
  double* buf = nullptr;
  if ((e = cudaMalloc(&buf, 256)) != cudaSuccess) return (int)e;
  const int iters = 1 << 15, blocks = sms * 8, threads = 256;
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0);
  cudaEventCreate(&e1);
  k_probe_dfma<<<blocks, threads>>>(buf, iters / 8); // warm-up
  float best = 1e30f;
  for (int rep = 0; rep < (reps > 0 ? reps : 3); ++rep) {
    cudaEventRecord(e0);
    k_probe_dfma<<<blocks, threads>>>(buf, iters);
    cudaEventRecord(e1);
    cudaEventSynchronize(e1);
    float ms = 0;
    cudaEventElapsedTime(&ms, e0, e1);
    if (ms < best) best = ms;
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(buf);
  if ((e = cudaGetLastError()) != cudaSuccess) return (int)e;
  *tflops = 2.0 * 8.0 * (double)iters * blocks * threads / (best * 1e-3) / 1e12;
  return 0;
}
