// Plain operator product on the panel kernels (panel.cuh): C[b] <- c1*A*B[b] + c2*C[b]  (eq. 1).
#include "panel_kernel.cuh"

namespace frb {

namespace {

template <typename T>
struct PlainArgs {
  PanelOp<T> op;
  PlainProducer<T> prod;
  PlainEpilogue<T> epi;
  long long npanels;
  int nbatch;
};

template <typename T, int NIT, int CX>
__global__ void __launch_bounds__(32 * panel_maxw<T>(NIT, CX)) k_panel_gemm(const __grid_constant__ PlainArgs<T> a) {
  extern __shared__ __align__(16) char panel_smem[];
  panel_mainloop<T, NIT, CX>(a.op, a.prod, a.epi, a.npanels, a.nbatch, panel_smem);
}

template <typename T, int NIT, int CX>
void launch_shape(const PlainArgs<T> &a, size_t smem, cudaStream_t s) {
  auto k = k_panel_gemm<T, NIT, CX>;
  static bool attr_done = false;
  static int occ = 1;
  static size_t attr_smem = 0;
  const int nthreads = 32 * a.op.WR * a.op.WC * a.op.NG;
  if (!attr_done || smem > attr_smem) {
    FR_CUDA_TRY(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)std::max(smem, attr_smem)));
    attr_smem = std::max(smem, attr_smem);
    attr_done = true;
  }
  FR_CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k, nthreads, smem));
  occ = std::max(1, std::min(occ, a.op.occ));
  const long long ntot = a.npanels * a.nbatch;
  const long long grid = std::min<long long>((ntot + a.op.NG - 1) / a.op.NG, (long long)device_sm_count() * occ);
  k<<<(unsigned)grid, nthreads, smem, s>>>(a);
  FR_CUDA_TRY(cudaGetLastError());
}

}  // namespace

template <typename T>
bool panel_gemm_build(PanelOp<T> &op, int M, int K, const double *A, int cand) {
  std::vector<KSource> srcs{KSource{K, 0, 1}};
  PackOptions opt;
  opt.min_ne = sizeof(T) == 8 ? 16 : 32;
  opt.max_ne = sizeof(T) == 8 ? 64 : 128;
  opt.cand = cand;
  return panel_op_build(op, M, K, A, srcs, opt, 150 * 1024);
}

template <typename T>
void panel_gemm_run(const PanelOp<T> &op, long long N, T c1, const T *B, long long ldb, long long bsB, T c2, T *C,
                    long long ldc, long long bsC, int nbatch, cudaStream_t s) {
  PlainArgs<T> a;
  a.op = op;
  const long long pw = (long long)PV * op.NE;
  ColMap cm{pw, op.NE, op.NE, N};
  a.prod = PlainProducer<T>();
  a.prod.src[0] = MatRef<T>{B, ldb, bsB};
  a.prod.src[1] = a.prod.src[0];
  a.prod.cm = cm;
  a.epi = PlainEpilogue<T>{C, ldc, bsC, cm, c1, c2};
  a.npanels = (N + pw - 1) / pw;
  a.nbatch = nbatch;
  const size_t smem = panel_smem_bytes(op);
#define FR_CASE(NIT_, CX_)                                     \
  if (op.NIT == NIT_ && op.CX == CX_) {                        \
    launch_shape<T, NIT_, CX_>(a, smem, s);                    \
    return;                                                    \
  }
  if constexpr (sizeof(T) == 8) {
    FR_PANEL_SHAPES_F64(FR_CASE)
  } else {
    FR_PANEL_SHAPES_F32(FR_CASE)
  }
#undef FR_CASE
  throw Error{FR_ESTATE, "panel_gemm_run: no kernel for this accumulator shape"};
}

template bool panel_gemm_build<double>(PanelOp<double> &, int, int, const double *, int);
template bool panel_gemm_build<float>(PanelOp<float> &, int, int, const double *, int);
template void panel_gemm_run<double>(const PanelOp<double> &, long long, double, const double *, long long, long long, double,
                                     double *, long long, long long, int, cudaStream_t);
template void panel_gemm_run<float>(const PanelOp<float> &, long long, float, const float *, long long, long long, float, float *,
                                    long long, long long, int, cudaStream_t);

}  // namespace frb
