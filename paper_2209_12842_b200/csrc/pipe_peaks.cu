// Measured issue rates of the plain SM pipes (roofline denominators for the ALU-bound rollout
// kernel; MEASURED_PEAKS.json has only HBM and tensor numbers).  Each kernel runs independent
// dependency chains of one instruction class, unrolled, on every SM with full occupancy, and the
// host reports lane-operations per second from CUDA events.
#include "../../include/ra_mppi.h"

#include <cuda_runtime.h>

#include <cstdint>

namespace {

constexpr int kChains = 8;      // independent chains per thread (ILP)
constexpr int kInner = 64;      // unrolled instructions per chain per outer iteration
constexpr int kThreads = 256;

__global__ void __launch_bounds__(kThreads) ffma_kernel(float* out, int iters, float a, float b) {
  float x[kChains];
#pragma unroll
  for (int i = 0; i < kChains; ++i) x[i] = (float)(threadIdx.x + i);
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int j = 0; j < kInner; ++j)
#pragma unroll
      for (int i = 0; i < kChains; ++i) x[i] = fmaf(x[i], a, b);
  }
  float s = 0.f;
#pragma unroll
  for (int i = 0; i < kChains; ++i) s += x[i];
  if (s == 123.456f) out[0] = s;
}

__global__ void __launch_bounds__(kThreads) imad_wide_kernel(float* out, int iters, uint32_t a) {
  uint32_t x[kChains];
#pragma unroll
  for (int i = 0; i < kChains; ++i) x[i] = threadIdx.x * 2654435761u + i;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int j = 0; j < kInner; ++j)
#pragma unroll
      for (int i = 0; i < kChains; ++i) {
        unsigned long long p;
        asm volatile("mul.wide.u32 %0, %1, %2;" : "=l"(p) : "r"(x[i] | 0x80000000u), "r"(a));  // IMAD.WIDE.U32
        x[i] = (uint32_t)(p >> 32);   // next input = high half: the wide form is kept, no extra add
      }
  }
  uint32_t s = 0;
#pragma unroll
  for (int i = 0; i < kChains; ++i) s ^= x[i];
  if (s == 0x12345u) out[0] = (float)s;
}

__global__ void __launch_bounds__(kThreads) lop3_kernel(float* out, int iters, uint32_t a, uint32_t b) {
  uint32_t x[kChains];
#pragma unroll
  for (int i = 0; i < kChains; ++i) x[i] = threadIdx.x * 2654435761u + i;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int j = 0; j < kInner; ++j)
#pragma unroll
      for (int i = 0; i < kChains; ++i)
        asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(x[i]) : "r"(a + j), "r"(b));   // 3-input XOR
  }
  uint32_t s = 0;
#pragma unroll
  for (int i = 0; i < kChains; ++i) s ^= x[i];
  if (s == 0x12345u) out[0] = (float)s;
}

__global__ void __launch_bounds__(kThreads) mufu_kernel(float* out, int iters) {
  float x[kChains];
#pragma unroll
  for (int i = 0; i < kChains; ++i) x[i] = 1.0f + 0.001f * (float)(threadIdx.x + i);
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int j = 0; j < kInner; ++j)
#pragma unroll
      for (int i = 0; i < kChains; ++i) asm volatile("lg2.approx.ftz.f32 %0, %0;" : "+f"(x[i]));
  }
  float s = 0.f;
#pragma unroll
  for (int i = 0; i < kChains; ++i) s += x[i];
  if (s == 123.456f) out[0] = s;
}

template <typename Launch>
bool time_kernel(Launch launch, double ops_per_launch, float* result) {
  cudaEvent_t a, b;
  if (cudaEventCreate(&a) != cudaSuccess || cudaEventCreate(&b) != cudaSuccess) return false;
  launch();  // warm-up
  float best = 1e30f;
  for (int rep = 0; rep < 5; ++rep) {
    cudaEventRecord(a);
    launch();
    cudaEventRecord(b);
    if (cudaEventSynchronize(b) != cudaSuccess) return false;
    float ms = 0.f;
    cudaEventElapsedTime(&ms, a, b);
    best = ms < best ? ms : best;
  }
  cudaEventDestroy(a);
  cudaEventDestroy(b);
  *result = (float)(ops_per_launch / (best * 1e-3) / 1e12);
  return cudaGetLastError() == cudaSuccess;
}

}  // namespace

extern "C" ra_status ra_mppi_measure_pipe_peaks(int32_t device, float* h_tera_lane_ops) {
  if (!h_tera_lane_ops) return RA_EINVAL;
  int n_dev = 0;
  if (cudaGetDeviceCount(&n_dev) != cudaSuccess || device < 0 || device >= n_dev) return RA_ECUDA;
  if (cudaSetDevice(device) != cudaSuccess) return RA_ECUDA;
  cudaDeviceProp prop{};
  if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) return RA_ECUDA;
  float* d_out = nullptr;
  if (cudaMalloc(&d_out, sizeof(float)) != cudaSuccess) return RA_ENOMEM;
  const int grid = prop.multiProcessorCount * 8;   // 2048 threads per SM
  const int iters = 256;
  const double ops = (double)grid * kThreads * iters * kInner * kChains;
  bool ok = true;
  ok = ok && time_kernel([&] { ffma_kernel<<<grid, kThreads>>>(d_out, iters, 1.0000001f, 1e-9f); }, ops, &h_tera_lane_ops[0]);
  ok = ok && time_kernel([&] { imad_wide_kernel<<<grid, kThreads>>>(d_out, iters, 0xD2511F53u); }, ops, &h_tera_lane_ops[1]);
  ok = ok && time_kernel([&] { lop3_kernel<<<grid, kThreads>>>(d_out, iters, 0x9E3779B9u, 0xBB67AE85u); }, ops, &h_tera_lane_ops[2]);
  ok = ok && time_kernel([&] { mufu_kernel<<<grid, kThreads>>>(d_out, iters); }, ops, &h_tera_lane_ops[3]);
  cudaFree(d_out);
  return ok ? RA_OK : RA_ECUDA;
}
