// Plain operator product on the panel kernels (panel.cuh): C[b] <- c1*A*B[b] + c2*C[b]  (eq. 1).
#include "panel_kernel.cuh"

namespace frb {

namespace {

template <typename T>
struct alignas(64) PlainArgs {
  TmaProducer<T> prod;
  PanelOp<T> op;
  PlainEpilogue<T> epi;
  long long npanels;
  int nbatch;
};

template <typename T, int NIT, int CX, bool STREAM, bool DYN>
__global__ void __launch_bounds__(32 * panel_maxw<T>(NIT, CX)) k_panel_gemm(const __grid_constant__ PlainArgs<T> a) {
  extern __shared__ __align__(1024) char panel_smem[];
  panel_mainloop<T, NIT, CX, TmaProducer<T>, PlainEpilogue<T>, true, STREAM, DYN>(a.op, a.prod, a.epi, a.npanels, a.nbatch, panel_smem);
}

}  // namespace

template <typename T>
bool panel_gemm_build(PanelOp<T> &op, int M, int K, const double *A, int cand, double drop_rel, int stream) {
  std::vector<KSource> srcs{KSource{K}};
  PackOptions opt;
  opt.min_ne = sizeof(T) == 8 ? 16 : 32;
  opt.max_ne = sizeof(T) == 8 ? 64 : 128;
  opt.cand = cand;
  opt.drop_rel = drop_rel;
  opt.stream = stream;
  return panel_op_build(op, M, K, A, srcs, opt, 150 * 1024);
}

template <typename T>
void panel_gemm_run(const PanelOp<T> &op, long long N, T c1, const T *B, long long ldb, long long bsB, T c2, T *C,
                    long long ldc, long long bsC, int nbatch, cudaStream_t s) {
  PlainArgs<T> a;
  a.op = op;
  a.op.pf_epi = 1;
  const long long pw = (long long)PV * op.NE;
  ColMap cm{pw, op.NE, op.NE, N};
  a.prod.tm[0] = tmap_plain(B, op.K, N, ldb, bsB, nbatch, op.NE, op.src_step[0]);
  a.prod.tm[1] = a.prod.tm[0];
  a.prod.plain = 1;
  a.epi = PlainEpilogue<T>{C, ldc, bsC, cm, c1, c2, (c1 == T(1) && c2 == T(0)) ? 1 : 0};
  a.npanels = (N + pw - 1) / pw;
  a.nbatch = nbatch;
  const bool units = panel_use_units(op);
#define FR_CASE(NIT_, CX_)                                                                        \
  if (op.NIT == NIT_ && op.CX == CX_) {                                                           \
    /* one warp group: the consumer warps take units from a counter (panel_kernel.cuh DYN) */     \
    if (units) {                                                                   \
      if (op.streamed()) panel_launch(k_panel_gemm<T, NIT_, CX_, true, true>, a, op, a.npanels * a.nbatch, s); \
      else panel_launch(k_panel_gemm<T, NIT_, CX_, false, true>, a, op, a.npanels * a.nbatch, s); \
    } else if (op.streamed()) panel_launch(k_panel_gemm<T, NIT_, CX_, true, false>, a, op, a.npanels * a.nbatch, s); \
    else panel_launch(k_panel_gemm<T, NIT_, CX_, false, false>, a, op, a.npanels * a.nbatch, s);  \
    return;                                                                                       \
  }
  if constexpr (sizeof(T) == 8) {
    FR_PANEL_SHAPES_F64(FR_CASE)
  } else {
    FR_PANEL_SHAPES_F32(FR_CASE)
  }
#undef FR_CASE
  throw Error{FR_ESTATE, "panel_gemm_run: no kernel for this accumulator shape"};
}

template bool panel_gemm_build<double>(PanelOp<double> &, int, int, const double *, int, double, int);
template bool panel_gemm_build<float>(PanelOp<float> &, int, int, const double *, int, double, int);
template void panel_gemm_run<double>(const PanelOp<double> &, long long, double, const double *, long long, long long, double,
                                     double *, long long, long long, int, cudaStream_t);
template void panel_gemm_run<float>(const PanelOp<float> &, long long, float, const float *, long long, long long, float, float *,
                                    long long, long long, int, cudaStream_t);

}  // namespace frb
