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
