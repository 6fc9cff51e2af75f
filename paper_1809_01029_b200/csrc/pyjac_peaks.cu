// Machine-peak microbenchmarks behind pyjac_measure_peak (include/pyjac.h): the denominators of the rooflines that
// bench.py reports (SURVEY.md section 8d "Peaks": measure the DFMA rate and a write-only stream, do not trust the
// datasheet).  Every figure is timed with CUDA events around `reps` back-to-back launches after one warm-up launch.
#include <cuda_runtime.h>

#include <cstdint>
#include <string>

#include "pyjac.h"

namespace {

constexpr int DFMA_CHAINS = 8;        // independent dependency chains per thread (DFMA latency 8 cycles, 2-cycle issue)
constexpr int DFMA_ITERS = 4096;

__global__ void __launch_bounds__(512) dfma_kernel(double* out, double a, double b) {
  double v[DFMA_CHAINS];
#pragma unroll
  for (int c = 0; c < DFMA_CHAINS; ++c) v[c] = (double)(threadIdx.x + c);
  for (int i = 0; i < DFMA_ITERS; ++i) {
#pragma unroll
    for (int c = 0; c < DFMA_CHAINS; ++c) v[c] = fma(v[c], a, b);
  }
  double s = 0.0;
#pragma unroll
  for (int c = 0; c < DFMA_CHAINS; ++c) s += v[c];
  if (s == 12345.678) out[0] = s;     // never true: keeps the chains alive
}

__global__ void __launch_bounds__(512) write_kernel(double2* p, size_t n) {
  const size_t stride = (size_t)gridDim.x * blockDim.x;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) __stcs(p + i, make_double2(0.0, 0.0));
}

__global__ void __launch_bounds__(512) read_kernel(const double2* p, size_t n, double* out) {
  const size_t stride = (size_t)gridDim.x * blockDim.x;
  double s = 0.0;
  size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  for (; i + 3 * stride < n; i += 4 * stride) {
    const double2 a = __ldcs(p + i), b = __ldcs(p + i + stride), c = __ldcs(p + i + 2 * stride), d = __ldcs(p + i + 3 * stride);
    s += a.x + a.y + b.x + b.y + c.x + c.y + d.x + d.y;
  }
  for (; i < n; i += stride) { const double2 a = __ldcs(p + i); s += a.x + a.y; }
  if (s == 12345.678) out[0] = s;
}

__global__ void __launch_bounds__(512) copy_kernel(const double2* src, double2* dst, size_t n) {
  const size_t stride = (size_t)gridDim.x * blockDim.x;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) __stcs(dst + i, __ldcs(src + i));
}

// every CTA sweeps the same L2-resident window `passes` times (L1 is bypassed: ld.global.cg)
__global__ void __launch_bounds__(512) l2_read_kernel(const double2* p, size_t n, int passes, double* out) {
  double s = 0.0;
  for (int q = 0; q < passes; ++q) {
    // CTAs start at different offsets so that they do not all hit one slice at a time
    const size_t off = ((size_t)blockIdx.x * 4099 + (size_t)q * 257) * blockDim.x % n;
    for (size_t j = threadIdx.x; j < n; j += 4 * blockDim.x) {
      size_t i0 = off + j, i1 = i0 + blockDim.x, i2 = i1 + blockDim.x, i3 = i2 + blockDim.x;
      i0 = i0 >= n ? i0 - n : i0; i1 = i1 >= n ? i1 - n : i1; i2 = i2 >= n ? i2 - n : i2; i3 = i3 >= n ? i3 - n : i3;
      const double2 a = __ldcg(p + i0), b = __ldcg(p + i1), c = __ldcg(p + i2), d = __ldcg(p + i3);
      s += a.x + a.y + b.x + b.y + c.x + c.y + d.x + d.y;
    }
  }
  if (s == 12345.678) out[0] = s;
}

// shared-memory load rate: conflict-free 16-byte loads (one wavefront per quarter-warp)
__global__ void __launch_bounds__(512) lds_kernel(double* out, int iters) {
  __shared__ double2 buf[2048];
  for (int i = threadIdx.x; i < 2048; i += blockDim.x) buf[i] = make_double2((double)i, 1.0);
  __syncthreads();
  double s = 0.0;
  int idx = threadIdx.x;
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int u = 0; u < 8; ++u) { const double2 v = buf[(idx + u * 256) & 2047]; s += v.x; idx += (int)v.y; }
  }
  if (s == 12345.678) out[0] = s;
}

thread_local std::string g_peak_err;

}  // namespace

extern "C" int pyjac_measure_peak(int kind, int cuda_device, int reps, double* value) {
  if (!value || reps < 1 || kind < 0 || kind > PYJAC_PEAK_LDS) return PYJAC_EINVAL;
  int prev = 0;
  cudaGetDevice(&prev);
  cudaError_t e = cudaSetDevice(cuda_device);
  if (e != cudaSuccess) return PYJAC_ECUDA;
  int n_sm = 0;
  cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, cuda_device);
  const size_t big = (size_t)4 << 30, window = (size_t)32 << 20;    // HBM streams: 4 GiB (>> L2); L2 window: 32 MiB
  void *a = nullptr, *b = nullptr;
  double* sink = nullptr;
  cudaEvent_t t0 = nullptr, t1 = nullptr;
  int rc = PYJAC_OK;
  double work = 0.0;           // bytes or DFMAs per launch
  auto launch = [&]() {
    switch (kind) {
      case PYJAC_PEAK_DFMA:
        dfma_kernel<<<n_sm * 4, 512>>>(sink, 0.999999, 1e-9);
        work = (double)n_sm * 4 * 512 * DFMA_CHAINS * DFMA_ITERS;
        break;
      case PYJAC_PEAK_HBM_WRITE:
        write_kernel<<<n_sm * 8, 512>>>((double2*)a, big / 16);
        work = (double)big;
        break;
      case PYJAC_PEAK_HBM_READ:
        read_kernel<<<n_sm * 8, 512>>>((const double2*)a, big / 16, sink);
        work = (double)big;
        break;
      case PYJAC_PEAK_HBM_COPY:
        copy_kernel<<<n_sm * 8, 512>>>((const double2*)a, (double2*)b, big / 16);
        work = 2.0 * (double)big;
        break;
      case PYJAC_PEAK_L2_READ:
        l2_read_kernel<<<n_sm * 4, 512>>>((const double2*)a, window / 16, 2, sink);
        work = (double)n_sm * 4 * 2 * (double)window;
        break;
      default:
        lds_kernel<<<n_sm * 2, 512>>>(sink, 2048);
        work = (double)n_sm * 2 * 512 * 2048.0 * 8 * 16;
        break;
    }
  };
  do {
    if ((e = cudaMalloc(&sink, 64)) != cudaSuccess) { rc = PYJAC_ECUDA; break; }
    const size_t na = kind == PYJAC_PEAK_L2_READ ? window : (kind >= PYJAC_PEAK_HBM_WRITE && kind <= PYJAC_PEAK_HBM_COPY ? big : 0);
    if (na && (e = cudaMalloc(&a, na)) != cudaSuccess) { rc = PYJAC_ENOMEM; break; }
    if (na && (e = cudaMemset(a, 0, na)) != cudaSuccess) { rc = PYJAC_ECUDA; break; }
    if (kind == PYJAC_PEAK_HBM_COPY && (e = cudaMalloc(&b, big)) != cudaSuccess) { rc = PYJAC_ENOMEM; break; }
    cudaEventCreate(&t0); cudaEventCreate(&t1);
    launch();                                     // warm-up
    if ((e = cudaDeviceSynchronize()) != cudaSuccess) { rc = PYJAC_ECUDA; break; }
    cudaEventRecord(t0);
    for (int r = 0; r < reps; ++r) launch();
    cudaEventRecord(t1);
    if ((e = cudaEventSynchronize(t1)) != cudaSuccess) { rc = PYJAC_ECUDA; break; }
    float ms = 0.f;
    cudaEventElapsedTime(&ms, t0, t1);
    *value = work * reps / (ms * 1e-3);
  } while (0);
  if (t0) cudaEventDestroy(t0);
  if (t1) cudaEventDestroy(t1);
  cudaFree(a); cudaFree(b); cudaFree(sink);
  cudaSetDevice(prev);
  return rc;
}
