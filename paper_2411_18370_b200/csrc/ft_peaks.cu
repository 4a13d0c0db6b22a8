// ft_measure_peaks: micro-benchmarks of the units that bound this library's kernels.
// MEASURED_PEAKS.json holds the HBM copy bandwidth and the bf16 GEMM rate only; the tile kernel is bound by the
// shared-memory data pipe and kernel K1 by the fp64 pipe, so their roofline denominators are measured here,
// on the same device, with the same instructions the kernels use (LDS.32, DFMA, F2I/I2F.F64, LDG through L2).
#include "ft_ctx.cuh"

namespace {

constexpr int PK_THREADS = 1024;

// conflict-free LDS.32: lane l of every warp reads word (l + 32 j + it) of a 32 KB array, 32 loads in flight
__global__ void __launch_bounds__(PK_THREADS)
pk_smem_kernel(float* __restrict__ out, int iters, long long* __restrict__ cycles) {
  __shared__ float buf[8192];
  for (int i = threadIdx.x; i < 8192; i += blockDim.x) buf[i] = (float)(i & 7);
  __syncthreads();
  const uint32_t base = (uint32_t)__cvta_generic_to_shared(buf);
  const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  float acc[8] = {0, 0, 0, 0, 0, 0, 0, 0};
  const long long t0 = clock64();
  for (int it = 0; it < iters; ++it) {
    const uint32_t ad = base + 4u * ((lane + 32u * ((warp + (uint32_t)it) & 31u)) & 8191u);
#pragma unroll
    for (int j = 0; j < 32; ++j) {
      float v;
      asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(ad + 128u * (uint32_t)j));
      acc[j & 7] += v;
    }
  }
  const long long t1 = clock64();
  float s = 0.f;
#pragma unroll
  for (int j = 0; j < 8; ++j) s += acc[j];
  if (s == -1.f) out[0] = s;
  if (threadIdx.x == 0 && blockIdx.x == 0) *cycles = t1 - t0;
}

__global__ void __launch_bounds__(PK_THREADS)
pk_dfma_kernel(double* __restrict__ out, int iters, double a, double b) {
  double x[8];
#pragma unroll
  for (int j = 0; j < 8; ++j) x[j] = (double)(threadIdx.x + j);
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int r = 0; r < 4; ++r)
#pragma unroll
      for (int j = 0; j < 8; ++j) x[j] = fma(x[j], a, b);
  }
  double s = 0.0;
#pragma unroll
  for (int j = 0; j < 8; ++j) s += x[j];
  if (s == -1.0) out[0] = s;
}

// F2I.F64 then I2F.F64 (the pair the canonical rounding k = rint(x), (double)k would cost per evaluation)
__global__ void __launch_bounds__(PK_THREADS)
pk_cvt_kernel(double* __restrict__ out, int iters, double b) {
  double x[8];
#pragma unroll
  for (int j = 0; j < 8; ++j) x[j] = (double)(threadIdx.x + j) + 0.25;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int r = 0; r < 4; ++r)
#pragma unroll
      for (int j = 0; j < 8; ++j) x[j] = (double)__double2int_rn(x[j]) + b;
  }
  double s = 0.0;
#pragma unroll
  for (int j = 0; j < 8; ++j) s += x[j];
  if (s == -1.0) out[0] = s;
}

// 16-byte loads that bypass L1 over a buffer resident in L2
__global__ void __launch_bounds__(PK_THREADS)
pk_l2_kernel(const uint4* __restrict__ buf, size_t n_vec, int passes, uint32_t* __restrict__ out) {
  uint32_t acc = 0;
  const size_t stride = (size_t)gridDim.x * blockDim.x;
  for (int p = 0; p < passes; ++p)
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n_vec; i += stride) {
      uint4 v;
      asm volatile("ld.global.cg.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(buf + i));
      acc += v.x ^ v.y ^ v.z ^ v.w;
    }
  if (acc == 0x12345678u) out[0] = acc;
}

}  // namespace

extern "C" int ft_measure_peaks(ft_ctx* c, ft_peaks* out) {
  if (!c || !out) return FT_ERR_ARG;
  if (!c->d.P) return ft_fail(c, FT_ERR_STATE, "ft_measure_peaks: handle not created");
  if (int rc = ft_enter(c)) return rc;
  cudaDeviceProp prop{};
  FT_CUDA(c, cudaGetDeviceProperties(&prop, c->device));
  const int n_sm = prop.multiProcessorCount;
  const size_t l2_bytes = (size_t)32 << 20;
  unsigned char* buf = nullptr;
  FT_CUDA(c, cudaMalloc(&buf, l2_bytes + 64));
  FT_CUDA(c, cudaMemsetAsync(buf, 1, l2_bytes + 64, c->stream));
  long long* cyc = reinterpret_cast<long long*>(buf + l2_bytes);
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  cudaEventCreate(&e0); cudaEventCreate(&e1);
  auto timed = [&](auto&& launch, int reps) {
    launch();   // warm-up
    float best = 1e30f;
    for (int r = 0; r < reps; ++r) {
      cudaEventRecord(e0, c->stream);
      launch();
      cudaEventRecord(e1, c->stream);
      cudaEventSynchronize(e1);
      float ms = 0.f;
      cudaEventElapsedTime(&ms, e0, e1);
      best = ms < best ? ms : best;
    }
    return (double)best * 1e-3;
  };
  const int grid = n_sm;   // one CTA of 1024 threads per SM (64 registers each: the register file holds one)
  {
    const int iters = 8000;
    const double s = timed([&] { pk_smem_kernel<<<grid, PK_THREADS, 0, c->stream>>>(reinterpret_cast<float*>(buf), iters, cyc); }, 3);
    out->smem_gbs = (double)grid * PK_THREADS * (double)iters * 32.0 * 4.0 / s / 1e9;
    long long h = 0;
    cudaMemcpy(&h, cyc, sizeof h, cudaMemcpyDeviceToHost);
    // one CTA per SM: block 0 ran for about the whole kernel
    out->sm_clock_mhz = (double)h / s / 1e6;
  }
  {
    const int iters = 4000;
    const double s = timed([&] { pk_dfma_kernel<<<grid, PK_THREADS, 0, c->stream>>>(reinterpret_cast<double*>(buf), iters, 1.0000001, 1e-9); }, 3);
    out->fp64_gflops = (double)grid * PK_THREADS * (double)iters * 32.0 * 2.0 / s / 1e9;
  }
  {
    const int iters = 1000;
    const double s = timed([&] { pk_cvt_kernel<<<grid, PK_THREADS, 0, c->stream>>>(reinterpret_cast<double*>(buf), iters, 0.25); }, 3);
    out->fp64_cvt_gops = (double)grid * PK_THREADS * (double)iters * 32.0 / s / 1e9;
  }
  {
    const int passes = 200;
    const double s = timed([&] { pk_l2_kernel<<<n_sm, PK_THREADS, 0, c->stream>>>(reinterpret_cast<const uint4*>(buf), l2_bytes / 16, passes,
                                                                                     reinterpret_cast<uint32_t*>(buf + l2_bytes + 32)); }, 3);
    out->l2_gbs = (double)l2_bytes * passes / s / 1e9;
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  const cudaError_t e = cudaStreamSynchronize(c->stream);
  cudaFree(buf);
  c->counters.kernel_launches += 16;
  if (e != cudaSuccess) return ft_fail(c, FT_ERR_CUDA, std::string("ft_measure_peaks: ") + cudaGetErrorString(e));
  return FT_OK;
}
