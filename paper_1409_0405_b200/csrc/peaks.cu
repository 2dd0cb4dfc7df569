// Measured roofline denominators (include/frb200.h fr_probe_peaks): register-resident FMA chains for the
// FP64 / FP32 pipes and a plain device-to-device copy for HBM.  SURVEY 8(d): "the builder measures both with a
// register-resident FMA-chain micro-benchmark at sustained clocks and uses the measured values".
#include "common.cuh"

namespace frb {
namespace {

template <typename T, int ILP>
__global__ void __launch_bounds__(256) k_fma_chain(T *out, int iters, T a, T b) {
  T x[ILP];
#pragma unroll
  for (int i = 0; i < ILP; ++i) x[i] = (T)(threadIdx.x + i) * (T)1e-3;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int i = 0; i < ILP; ++i) x[i] = fma(x[i], a, b);
  }
  T s = 0;
#pragma unroll
  for (int i = 0; i < ILP; ++i) s += x[i];
  if (s == (T)123456.789) out[0] = s;   // never true; keeps the chain alive
}

// FP64 tensor pipe: mma.sync.m8n8k4.f64 chains, NACC independent accumulators per warp (512 flops per instruction and warp)
template <int NACC>
__global__ void __launch_bounds__(256) k_dmma_chain(double *out, int iters, double a, double b) {
  double c[NACC][2];
#pragma unroll
  for (int i = 0; i < NACC; ++i) c[i][0] = c[i][1] = (double)(threadIdx.x + i) * 1e-3;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int i = 0; i < NACC; ++i)
      asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                   : "+d"(c[i][0]), "+d"(c[i][1])
                   : "d"(a), "d"(b));
  }
  double s = 0;
#pragma unroll
  for (int i = 0; i < NACC; ++i) s += c[i][0] + c[i][1];
  if (s == 123456.789) out[0] = s;   // never true; keeps the chain alive
}

double dmma_tflops() {
  constexpr int NACC = 8;
  const int blocks = device_sm_count() * 2, iters = 1 << 13;
  double *d = nullptr;
  FR_CUDA_TRY(cudaMalloc(&d, 64));
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0);
  cudaEventCreate(&e1);
  double best = 0;
  for (int rep = 0; rep < 6; ++rep) {
    cudaEventRecord(e0);
    k_dmma_chain<NACC><<<blocks, 256>>>(d, iters, 1e-3, 1e-3);
    cudaEventRecord(e1);
    FR_CUDA_TRY(cudaEventSynchronize(e1));
    float ms = 0;
    cudaEventElapsedTime(&ms, e0, e1);
    const double fl = 512.0 * NACC * (double)iters * 8.0 * blocks;   // 8 warps per block
    if (rep > 0) best = std::max(best, fl / (ms * 1e-3) / 1e12);
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(d);
  return best;
}

// FP32 alternatives (fr_probe_fp32_paths): packed fma.rn.f32x2 chains, FFMA / FFMA2 chains with NINT integer multiply-adds beside the
// 16 FMAs of an iteration (what address arithmetic and loop control cost the multiply loops), and the legacy TF32 tensor path.
template <bool PACKED, int NINT>
__global__ void __launch_bounds__(256) k_fp32_mixed(float *out, int iters, float a, float b) {
  constexpr int ILP = 16;
  float x[ILP];
#pragma unroll
  for (int i = 0; i < ILP; ++i) x[i] = (float)(threadIdx.x + i) * 1e-3f;
  unsigned long long xp[ILP / 2], ap, bp;
  asm("mov.b64 %0, {%1, %1};" : "=l"(ap) : "f"(a));
  asm("mov.b64 %0, {%1, %1};" : "=l"(bp) : "f"(b));
#pragma unroll
  for (int i = 0; i < ILP / 2; ++i) asm("mov.b64 %0, {%1, %2};" : "=l"(xp[i]) : "f"(x[2 * i]), "f"(x[2 * i + 1]));
  unsigned z = threadIdx.x;
  for (int it = 0; it < iters; ++it) {
    if (PACKED) {
#pragma unroll
      for (int i = 0; i < ILP / 2; ++i) asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(xp[i]) : "l"(ap), "l"(bp));
    } else {
#pragma unroll
      for (int i = 0; i < ILP; ++i) x[i] = fmaf(x[i], a, b);
    }
#pragma unroll
    for (int e = 0; e < NINT; ++e) z = z * 1664525u + 1013904223u;
  }
  float s = (float)z;
#pragma unroll
  for (int i = 0; i < ILP / 2; ++i) {
    float lo, hi;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(xp[i]));
    s += lo + hi + x[2 * i] + x[2 * i + 1];
  }
  if (s == 123456.789f) out[0] = s;   // never true; keeps the chains alive
}

template <int NACC>
__global__ void __launch_bounds__(256) k_tf32_mma_chain(float *out, int iters) {
  float c[NACC][4];
#pragma unroll
  for (int i = 0; i < NACC; ++i) c[i][0] = c[i][1] = c[i][2] = c[i][3] = 0.f;
  const unsigned a0 = __float_as_uint(1e-3f * threadIdx.x), a1 = __float_as_uint(2e-3f), b0 = __float_as_uint(3e-3f), b1 = __float_as_uint(1e-3f);
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int i = 0; i < NACC; ++i)
      asm volatile("mma.sync.aligned.m16n8k8.row.col.f32.tf32.tf32.f32 {%0,%1,%2,%3}, {%4,%5,%4,%5}, {%6,%7}, {%0,%1,%2,%3};\n"
                   : "+f"(c[i][0]), "+f"(c[i][1]), "+f"(c[i][2]), "+f"(c[i][3])
                   : "r"(a0), "r"(a1), "r"(b0), "r"(b1));
  }
  float s = 0;
#pragma unroll
  for (int i = 0; i < NACC; ++i) s += c[i][0] + c[i][1] + c[i][2] + c[i][3];
  if (s == 123456.789f) out[0] = s;
}

// best of 5 launches after a warm-up; `flops` per launch
template <typename L>
double probe_tflops(L &&launch, double flops) {
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0);
  cudaEventCreate(&e1);
  double best = 0;
  for (int rep = 0; rep < 6; ++rep) {
    cudaEventRecord(e0);
    launch();
    cudaEventRecord(e1);
    const cudaError_t st = cudaEventSynchronize(e1);
    if (st != cudaSuccess) {
      cudaEventDestroy(e0);
      cudaEventDestroy(e1);
      throw Error{FR_ECUDA, std::string("probe: ") + cudaGetErrorString(st)};
    }
    float ms = 0;
    cudaEventElapsedTime(&ms, e0, e1);
    if (rep > 0) best = std::max(best, flops / (ms * 1e-3) / 1e12);
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  return best;
}

void fp32_paths(double *out4) {
  float *d = nullptr;
  FR_CUDA_TRY(cudaMalloc(&d, 64));
  const int blocks = device_sm_count() * 8, iters = 1 << 14;
  const double fl = 2.0 * 16 * (double)iters * 256.0 * blocks;
  try {
    out4[0] = probe_tflops([&] { k_fp32_mixed<true, 0><<<blocks, 256>>>(d, iters, 0.999f, 1e-4f); }, fl);
    out4[1] = probe_tflops([&] { k_fp32_mixed<false, 8><<<blocks, 256>>>(d, iters, 0.999f, 1e-4f); }, fl);
    out4[2] = probe_tflops([&] { k_fp32_mixed<true, 8><<<blocks, 256>>>(d, iters, 0.999f, 1e-4f); }, fl);
    const int tb = device_sm_count() * 2;
    out4[3] = probe_tflops([&] { k_tf32_mma_chain<8><<<tb, 256>>>(d, iters); }, 2.0 * 16 * 8 * 8 * 8.0 * (double)iters * 8.0 * tb);
  } catch (...) {
    cudaFree(d);
    throw;
  }
  cudaFree(d);
}

__global__ void __launch_bounds__(256) k_copy(const float4 *__restrict__ in, float4 *__restrict__ out, size_t n) {
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) out[i] = in[i];
}

template <typename T>
double fma_tflops() {
  constexpr int ILP = 16;
  const int sms = device_sm_count();
  const int blocks = sms * 8, iters = 1 << 14;
  T *d = nullptr;
  FR_CUDA_TRY(cudaMalloc(&d, 64));
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0);
  cudaEventCreate(&e1);
  double best = 0;
  for (int rep = 0; rep < 6; ++rep) {
    cudaEventRecord(e0);
    k_fma_chain<T, ILP><<<blocks, 256>>>(d, iters, (T)0.999, (T)1e-4);
    cudaEventRecord(e1);
    FR_CUDA_TRY(cudaEventSynchronize(e1));
    float ms = 0;
    cudaEventElapsedTime(&ms, e0, e1);
    const double fl = 2.0 * ILP * (double)iters * 256.0 * blocks;
    if (rep > 0) best = std::max(best, fl / (ms * 1e-3) / 1e12);
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(d);
  return best;
}

double copy_gbs() {
  const size_t bytes = (size_t)1 << 30;
  float4 *a = nullptr, *b = nullptr;
  FR_CUDA_TRY(cudaMalloc(&a, bytes));
  if (cudaMalloc(&b, bytes) != cudaSuccess) {
    cudaFree(a);
    throw Error{FR_ENOMEM, "fr_probe_peaks: cannot allocate copy buffers"};
  }
  cudaMemset(a, 1, bytes);
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0);
  cudaEventCreate(&e1);
  double best = 0;
  for (int rep = 0; rep < 8; ++rep) {
    cudaEventRecord(e0);
    k_copy<<<device_sm_count() * 16, 256>>>(a, b, bytes / 16);
    cudaEventRecord(e1);
    cudaEventSynchronize(e1);
    float ms = 0;
    cudaEventElapsedTime(&ms, e0, e1);
    if (rep > 1) best = std::max(best, 2.0 * bytes / (ms * 1e-3) / 1e9);
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(a);
  cudaFree(b);
  return best;
}

}  // namespace
}  // namespace frb

extern "C" fr_status fr_probe_dmma(double *fp64_tensor_tflops) {
  try {
    int n = 0;
    if (cudaGetDeviceCount(&n) != cudaSuccess || n <= 0) return FR_ECUDA;
    if (fp64_tensor_tflops) *fp64_tensor_tflops = frb::dmma_tflops();
    return FR_OK;
  } catch (const frb::Error &e) {
    return e.st;
  } catch (...) {
    return FR_ESTATE;
  }
}

extern "C" fr_status fr_probe_fp32_paths(double *ffma2_tflops, double *ffma_mixed_tflops, double *ffma2_mixed_tflops, double *tf32_mma_tflops) {
  try {
    int n = 0;
    if (cudaGetDeviceCount(&n) != cudaSuccess || n <= 0) return FR_ECUDA;
    double v[4];
    frb::fp32_paths(v);
    if (ffma2_tflops) *ffma2_tflops = v[0];
    if (ffma_mixed_tflops) *ffma_mixed_tflops = v[1];
    if (ffma2_mixed_tflops) *ffma2_mixed_tflops = v[2];
    if (tf32_mma_tflops) *tf32_mma_tflops = v[3];
    return FR_OK;
  } catch (const frb::Error &e) {
    return e.st;
  } catch (...) {
    return FR_ESTATE;
  }
}

extern "C" fr_status fr_probe_peaks(double *fp64_tflops, double *fp32_tflops, double *copy_gbs_out) {
  try {
    int n = 0;
    if (cudaGetDeviceCount(&n) != cudaSuccess || n <= 0) return FR_ECUDA;
    if (fp64_tflops) *fp64_tflops = frb::fma_tflops<double>();
    if (fp32_tflops) *fp32_tflops = frb::fma_tflops<float>();
    if (copy_gbs_out) *copy_gbs_out = frb::copy_gbs();
    return FR_OK;
  } catch (const frb::Error &e) {
    return e.st;
  } catch (...) {
    return FR_ESTATE;
  }
}
