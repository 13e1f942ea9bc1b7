// cdz_peak.cu -- register-resident fp64 / fp32 issue-rate microbenchmarks (libcdz_peak.so: used by bench.py only, NOT part of the
// product ABI of include/cdz.h).
// MEASURED_PEAKS.json holds HBM and bf16 numbers only; the roofline of the fp64 split-point contraction needs the
// fp64 vector (DFMA) and tensor (mma.sync m8n8k4 f64, "DMMA") peaks of the same GPU under the same clocks.
#include <cuda_runtime.h>

#include <algorithm>

namespace {
__global__ void __launch_bounds__(512) peak_dfma(double* out, int iters) {
  double a[16];
  const double x = 1.0 + 1e-9 * threadIdx.x, y = 1e-9;
#pragma unroll
  for (int k = 0; k < 16; ++k) a[k] = k + threadIdx.x;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int k = 0; k < 16; ++k) a[k] = fma(a[k], x, y);
  }
  double s = 0;
#pragma unroll
  for (int k = 0; k < 16; ++k) s += a[k];
  out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}
__global__ void __launch_bounds__(512) peak_dmma(double* out, int iters) {
  double c[8][2];
  const double a = 1.0 + 1e-9 * threadIdx.x, b = 1e-9 * threadIdx.x;
#pragma unroll
  for (int k = 0; k < 8; ++k) c[k][0] = c[k][1] = k;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int k = 0; k < 8; ++k)
      asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                   : "+d"(c[k][0]), "+d"(c[k][1])
                   : "d"(a), "d"(b));
  }
  double s = 0;
#pragma unroll
  for (int k = 0; k < 8; ++k) s += c[k][0] + c[k][1];
  out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}
__global__ void __launch_bounds__(512) peak_ffma(float* out, int iters) {
  float a[16];
  const float x = 1.0f + 1e-6f * threadIdx.x, y = 1e-6f;
#pragma unroll
  for (int k = 0; k < 16; ++k) a[k] = k + threadIdx.x;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int k = 0; k < 16; ++k) a[k] = fmaf(a[k], x, y);
  }
  float s = 0;
#pragma unroll
  for (int k = 0; k < 16; ++k) s += a[k];
  out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}
}  // namespace

// kind 0 = fp64 FMA, 1 = fp64 mma.sync m8n8k4, 2 = fp32 FMA; TFLOP/s on the current device (best of 3 after one warm-up).
// Returns 0 on success, -1 on a bad argument, -3 on a CUDA error.
extern "C" int cdz_peak_measure(int kind, double* tflops_out) {
  if (!tflops_out || kind < 0 || kind > 2) return -1;
  cudaDeviceProp prop;
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) return -3;
  const int threads = 512, blocks = prop.multiProcessorCount * 4, iters = 20000;
  double* out = nullptr;
  if (cudaMalloc((void**)&out, sizeof(double) * threads * blocks) != cudaSuccess) return -3;
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0);
  cudaEventCreate(&e1);
  double best = 0;
  for (int rep = 0; rep < 4; ++rep) {
    cudaEventRecord(e0);
    if (kind == 0) peak_dfma<<<blocks, threads>>>(out, iters);
    else if (kind == 1) peak_dmma<<<blocks, threads>>>(out, iters);
    else peak_ffma<<<blocks, threads>>>((float*)out, iters);
    cudaEventRecord(e1);
    cudaEventSynchronize(e1);
    float ms = 0;
    cudaEventElapsedTime(&ms, e0, e1);
    const double flop = kind == 1 ? 2.0 * blocks * (threads / 32) * 8.0 * 256.0 * iters
                                  : 2.0 * blocks * threads * 16.0 * iters;
    if (rep > 0) best = std::max(best, flop / ms / 1e9);
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(out);
  if (cudaGetLastError() != cudaSuccess) return -3;
  *tflops_out = best;
  return 0;
}

// ---- dependency-latency floor of the blocked wavefront (SURVEY.md 8d "the third number") -----------------------------------
namespace {
__global__ void empty_kernel() {}
__global__ void __launch_bounds__(512) barrier_rounds(int rounds, int* sink) {
  __shared__ int s;
  if (threadIdx.x == 0) s = 0;
  for (int r = 0; r < rounds; ++r) {
    __syncthreads();
    if ((int)threadIdx.x == (r & 511)) s += r;  // a dependent shared-memory update per round, as the phases of the cell kernel have
  }
  __syncthreads();
  if (threadIdx.x == 0) sink[blockIdx.x] = s;
}
}  // namespace

// Average microseconds per launch of `count` dependent empty kernels on one stream (launch + completion chain).
extern "C" int cdz_peak_launch_us(int count, double* us_out) {
  if (!us_out || count <= 0) return -1;
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0);
  cudaEventCreate(&e1);
  for (int k = 0; k < 64; ++k) empty_kernel<<<1, 32>>>();
  cudaEventRecord(e0);
  for (int k = 0; k < count; ++k) empty_kernel<<<148, 128>>>();
  cudaEventRecord(e1);
  cudaEventSynchronize(e1);
  float ms = 0;
  cudaEventElapsedTime(&ms, e0, e1);
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  if (cudaGetLastError() != cudaSuccess) return -3;
  *us_out = 1e3 * ms / count;
  return 0;
}

// Microseconds per __syncthreads round of a 512-thread CTA (one CTA per SM, `rounds` dependent rounds).
extern "C" int cdz_peak_barrier_us(int rounds, double* us_out) {
  if (!us_out || rounds <= 0) return -1;
  int* sink = nullptr;
  if (cudaMalloc((void**)&sink, sizeof(int) * 148) != cudaSuccess) return -3;
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0);
  cudaEventCreate(&e1);
  barrier_rounds<<<148, 512>>>(rounds, sink);
  cudaEventRecord(e0);
  barrier_rounds<<<148, 512>>>(rounds, sink);
  cudaEventRecord(e1);
  cudaEventSynchronize(e1);
  float ms = 0;
  cudaEventElapsedTime(&ms, e0, e1);
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(sink);
  if (cudaGetLastError() != cudaSuccess) return -3;
  *us_out = 1e3 * ms / rounds;
  return 0;
}
