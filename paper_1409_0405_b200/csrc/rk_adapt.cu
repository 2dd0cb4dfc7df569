// Error estimate of the embedded pair RK4(3)5[2R+] and its norm (include/frb200.h fr_rk_adaptive_run).
//
// The stage kernels keep  X_i = X_{i-1} + dt b_i K_i  and  Y_i = X_{i-1} + dt a_i K_i  (a_5 = 0, so Y_5 = X_4), hence
//   dt (b_i - bhat_i) K_i = g_i (Y_i - X_i),   g_i = (b_i - bhat_i) / (a_i - b_i):
// the error register is accumulated from the two registers a stage has just written, without touching the fused stage kernels
// and without forming E as a small difference of O(|u|) quantities.  The last stage's contribution is folded into the norm
// kernel.  The norm is reduced in two passes with a fixed grid and a fixed summation tree: bit-reproducible, FP64 sums.
#include "kernels.cuh"

namespace frb {

namespace {

constexpr int ERR_BLOCK = 256;

template <typename T>
__global__ void __launch_bounds__(ERR_BLOCK) k_rk_err_accum(T *__restrict__ E, const T *__restrict__ Y, const T *__restrict__ X, T g,
                                                            int first, long long n) {
  const long long stride = (long long)gridDim.x * ERR_BLOCK;
  for (long long i = (long long)blockIdx.x * ERR_BLOCK + threadIdx.x; i < n; i += stride) {
    const T d = g * (Y[i] - X[i]);
    E[i] = first ? d : E[i] + d;
  }
}

__device__ __forceinline__ double block_sum(double v, double *sh) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
  const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
  if (l == 0) sh[w] = v;
  __syncthreads();
  double s = 0;
  if (threadIdx.x == 0)
    for (int i = 0; i < ERR_BLOCK / 32; ++i) s += sh[i];
  return s;   // valid in thread 0
}

// partial[block] = sum over this block's entries of ((E + g (Y - X)) / (atol + rtol max(|U0|, |X|)))^2 ; tol = {atol, rtol} (device)
template <typename T>
__global__ void __launch_bounds__(ERR_BLOCK) k_rk_err_norm(const T *__restrict__ E, const T *__restrict__ Y, const T *__restrict__ X,
                                                           const T *__restrict__ U0, T g, const double *__restrict__ tol,
                                                           long long n, double *__restrict__ partial) {
  __shared__ double sh[ERR_BLOCK / 32];
  const double atol = tol[0], rtol = tol[1];
  const long long stride = (long long)gridDim.x * ERR_BLOCK;
  double acc = 0;
  for (long long i = (long long)blockIdx.x * ERR_BLOCK + threadIdx.x; i < n; i += stride) {
    const T x = X[i];
    const double e = (double)(E[i] + g * (Y[i] - x));
    const double sc = atol + rtol * fmax(fabs((double)U0[i]), fabs((double)x));
    const double r = e / sc;
    acc += r * r;
  }
  const double s = block_sum(acc, sh);
  if (threadIdx.x == 0) partial[blockIdx.x] = s;
}

__global__ void __launch_bounds__(ERR_BLOCK) k_rk_err_final(const double *__restrict__ partial, int n, double *__restrict__ out) {
  __shared__ double sh[ERR_BLOCK / 32];
  double acc = 0;
  for (int i = threadIdx.x; i < n; i += ERR_BLOCK) acc += partial[i];
  const double s = block_sum(acc, sh);
  if (threadIdx.x == 0) out[0] = s;
}

}  // namespace

int rk_err_blocks() { return 8 * device_sm_count(); }

template <typename T>
int launch_rk_err_accum(T *E, const T *Y, const T *X, double g, int first, long long n, cudaStream_t s) {
  const int nb = (int)std::min<long long>(rk_err_blocks(), (n + ERR_BLOCK - 1) / ERR_BLOCK);
  k_rk_err_accum<T><<<nb, ERR_BLOCK, 0, s>>>(E, Y, X, (T)g, first, n);
  FR_CUDA_TRY(cudaGetLastError());
  return 1;
}

template <typename T>
int launch_rk_err_norm(const T *E, const T *Y, const T *X, const T *U0, double g, const double *tol_dev, long long n,
                       double *partial, cudaStream_t s) {
  // always the full grid: blocks beyond the data write 0, so the final pass sums a fixed number of partials
  k_rk_err_norm<T><<<rk_err_blocks(), ERR_BLOCK, 0, s>>>(E, Y, X, U0, (T)g, tol_dev, n, partial);
  FR_CUDA_TRY(cudaGetLastError());
  return 1;
}

int launch_rk_err_final(const double *partial, int n, double *out, cudaStream_t s) {
  k_rk_err_final<<<1, ERR_BLOCK, 0, s>>>(partial, n, out);
  FR_CUDA_TRY(cudaGetLastError());
  return 1;
}

template int launch_rk_err_accum<double>(double *, const double *, const double *, double, int, long long, cudaStream_t);
template int launch_rk_err_accum<float>(float *, const float *, const float *, double, int, long long, cudaStream_t);
template int launch_rk_err_norm<double>(const double *, const double *, const double *, const double *, double, const double *,
                                        long long, double *, cudaStream_t);
template int launch_rk_err_norm<float>(const float *, const float *, const float *, const float *, double, const double *, long long,
                                       double *, cudaStream_t);

}  // namespace frb
