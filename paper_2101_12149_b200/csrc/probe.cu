// On-chip ceilings measured on the device the library runs on (include/pic.h, pic_probe_peaks): the
// paper's roofline method uses MEASURED ceilings (Fig. 2, ref [27]); the
// particle kernels of this library are bound on chip (fp64 pipe, shared-memory bandwidth), and those
// two roofs are in no driver-written file. Each probe is a register-resident loop with enough
// independent chains and resident warps to fill its unit; nothing here is on the PIC path.
#include <algorithm>
#include <cmath>

#include "pic.h"

namespace pic {
namespace {

constexpr int kProbeThreads = 256;
constexpr int kProbeIters = 4096;

// 8 independent DFMA chains per thread
__global__ void __launch_bounds__(kProbeThreads) k_probe_dfma(double* out, double b, double c) {
  double a[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) a[i] = (double)(threadIdx.x + i);
#pragma unroll 1
  for (int it = 0; it < kProbeIters; ++it) {
#pragma unroll
    for (int i = 0; i < 8; ++i) a[i] = fma(a[i], b, c);
  }
  double s = 0;
#pragma unroll
  for (int i = 0; i < 8; ++i) s += a[i];
  if (s == 123.456) out[0] = s;   // never true: keeps the chains alive
}

// 16 independent FFMA chains per thread
__global__ void __launch_bounds__(kProbeThreads) k_probe_ffma(float* out, float b, float c) {
  float a[16];
#pragma unroll
  for (int i = 0; i < 16; ++i) a[i] = (float)(threadIdx.x + i);
#pragma unroll 1
  for (int it = 0; it < kProbeIters; ++it) {
#pragma unroll
    for (int i = 0; i < 16; ++i) a[i] = fmaf(a[i], b, c);
  }
  float s = 0;
#pragma unroll
  for (int i = 0; i < 16; ++i) s += a[i];
  if (s == 123.456f) out[0] = s;
}

// 4 independent accumulators of mma.sync.m8n8k4.f64 per warp (the instruction k_deposit_mma issues)
__global__ void __launch_bounds__(kProbeThreads) k_probe_dmma(double* out, double a, double b) {
  double c[4][2];
#pragma unroll
  for (int i = 0; i < 4; ++i) { c[i][0] = threadIdx.x; c[i][1] = i; }
#pragma unroll 1
  for (int it = 0; it < kProbeIters; ++it) {
#pragma unroll
    for (int i = 0; i < 4; ++i)
      asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                   : "+d"(c[i][0]), "+d"(c[i][1])
                   : "d"(a), "d"(b));
  }
  double s = 0;
#pragma unroll
  for (int i = 0; i < 4; ++i) s += c[i][0] + c[i][1];
  if (s == 123.456) out[0] = s;
}

// conflict-free 64-bit shared-memory loads (the access width of the fp64 gather), 8 per iteration
__global__ void __launch_bounds__(kProbeThreads) k_probe_lds64(double* out, int stride) {
  __shared__ unsigned long long buf[4096];   // 32 KB
  for (int i = threadIdx.x; i < 4096; i += blockDim.x) buf[i] = (unsigned long long)i * 0x9E3779B97F4A7C15ull;
  __syncthreads();
  unsigned long long s0 = 0, s1 = 0, s2 = 0, s3 = 0;   // integer accumulation: the fp64 pipe stays out of it
  int idx = threadIdx.x;
#pragma unroll 1
  for (int it = 0; it < kProbeIters; ++it) {
    const volatile unsigned long long* p = buf;
    s0 ^= p[(idx) & 4095];           s1 ^= p[(idx + 256) & 4095];
    s2 ^= p[(idx + 512) & 4095];     s3 ^= p[(idx + 768) & 4095];
    s0 ^= p[(idx + 1024) & 4095];    s1 ^= p[(idx + 1280) & 4095];
    s2 ^= p[(idx + 1536) & 4095];    s3 ^= p[(idx + 1792) & 4095];
    idx += stride;
  }
  const unsigned long long s = s0 ^ s1 ^ s2 ^ s3;
  if (s == 0x123456789ull) out[0] = (double)s;
}

}  // namespace
}  // namespace pic

extern "C" int pic_probe_peaks(void* cuda_stream, double seconds_per_probe, double* out) {
  using namespace pic;
  if (!out || !(seconds_per_probe >= 0) || !std::isfinite(seconds_per_probe)) return PIC_ERR_INVALID_ARG;
  for (int i = 0; i < PIC_NPROBE; ++i) out[i] = 0.0;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  int dev = 0, sms = 0, clk_khz = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) {
    cudaGetLastError();
    return PIC_ERR_CUDA;
  }
  cudaDeviceGetAttribute(&clk_khz, cudaDevAttrClockRate, dev);
  double* scratch = nullptr;
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  if (cudaMalloc(&scratch, 64) != cudaSuccess || cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) {
    cudaGetLastError();
    if (scratch) cudaFree(scratch);
    if (e0) cudaEventDestroy(e0);
    return PIC_ERR_CUDA;
  }
  const int grid = sms * 8;   // 8 CTAs of 256 threads per SM: every warp slot taken
  const double threads = (double)grid * kProbeThreads;
  // work of ONE launch of each probe
  const double work[PIC_NPROBE] = {
      threads * kProbeIters * 8 * 2.0,                 // DFMA flop
      threads / 32 * kProbeIters * 4 * 512.0,          // DMMA flop (m8n8k4 = 256 FMA)
      threads * kProbeIters * 8 * 8.0,                 // shared-memory bytes
      threads * kProbeIters * 16 * 2.0,                // FFMA flop
  };
  auto launch = [&](int which) {
    switch (which) {
      case PIC_PROBE_FP64_FMA_TFLOPS: k_probe_dfma<<<grid, kProbeThreads, 0, st>>>(scratch, 1.0000001, 1e-9); break;
      case PIC_PROBE_FP64_MMA_TFLOPS: k_probe_dmma<<<grid, kProbeThreads, 0, st>>>(scratch, 1.0000001, 1e-9); break;
      case PIC_PROBE_SMEM_TBS: k_probe_lds64<<<grid, kProbeThreads, 0, st>>>(scratch, 32); break;
      default: k_probe_ffma<<<grid, kProbeThreads, 0, st>>>((float*)scratch, 1.0000001f, 1e-9f); break;
    }
  };
  int rc = PIC_OK;
  for (int which = 0; which < 4 && rc == PIC_OK; ++which) {
    launch(which);   // warm-up
    double best = 0.0, total_s = 0.0;
    int reps = 0;
    while (reps < 3 || total_s < seconds_per_probe) {
      cudaEventRecord(e0, st);
      launch(which);
      cudaEventRecord(e1, st);
      if (cudaEventSynchronize(e1) != cudaSuccess) { rc = PIC_ERR_CUDA; break; }
      float ms = 0;
      cudaEventElapsedTime(&ms, e0, e1);
      if (ms > 0) best = std::max(best, work[which] / (ms * 1e-3) / 1e12);
      total_s += ms * 1e-3;
      if (++reps > 100000) break;
    }
    out[which] = best;
  }
  out[PIC_PROBE_SM_COUNT] = sms;
  out[PIC_PROBE_SM_CLOCK_MHZ] = clk_khz / 1e3;
  if (cudaGetLastError() != cudaSuccess) rc = PIC_ERR_CUDA;
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(scratch);
  return rc;
}
