// Fused panel kernels (fusion targets F-A and F-B of SURVEY 7.2):
//   fused_div : S6 + S8 + S9 + S10   dudt = -(1/|J|) [ M132 F~(U,G) + M3 D ]  (+ Runge-Kutta stage update)
//               the transformed flux F~ is formed in shared memory from the U, G and metric panels and never touches HBM;
//   fused_grad: S3 + S4              G_i = (1/|J|) sum_alpha S[alpha][i] ( [M460 | M6] [U; C] )_alpha
//               the three alpha components of a solution point sit in one thread (triple packing), so the transform to
//               physical gradients happens in registers.
// Both run on the persistent panel main loop (panel_kernel.cuh) with the operator resident in shared memory.
#include "kernels.cuh"
#include "panel_kernel.cuh"
#include "physics.cuh"

namespace frb {

namespace {

// ------------------------------------------------------------------------------------------------ fused_div
template <typename T>
struct FluxProducer {
  const T *u, *g, *d;       // state [Nu][5][ld]; gradients [3][Nu][5][ld] (NS only); common flux D [Nf][5][ld]
  const T *smats;           // [9][Nu][ld] or [9][ld]
  long long ld, neles;
  int nupts, curved;
  PhysParams<T> ph;
  static constexpr bool kTransform = true;

  __device__ __forceinline__ void issue(const ChunkDesc &cd, long long, long long pl, T *stage, int LDB, int NE, int tid,
                                        int nthreads) const {
    const long long e0 = pl * NE;
    if (cd.kind == KIND_PLAIN) {
      cp_rows5(stage, LDB, NE, d + (long long)cd.row0 * 5 * ld + e0, 5 * ld, ld, cd.nrows, tid, nthreads);
      return;
    }
    const int n = cd.nrows;
    if (ph.ns) {
#pragma unroll
      for (int a = 0; a < 3; ++a)
        cp_rows5(stage + a * n * LDB, LDB, NE, g + ((long long)a * nupts + cd.row0) * 5 * ld + e0, 5 * ld, ld, n, tid, nthreads);
    }
    cp_rows5(stage + 3 * n * LDB, LDB, NE, u + (long long)cd.row0 * 5 * ld + e0, 5 * ld, ld, n, tid, nthreads);
    T *sm = stage + 4 * n * LDB;
    if (curved) {
#pragma unroll
      for (int a = 0; a < 9; ++a)
        cp_rows1(sm + a * n * NE, NE, smats + ((long long)a * nupts + cd.row0) * ld + e0, ld, n, tid, nthreads);
    } else {
      cp_rows1(sm, NE, smats + e0, ld, 9, tid, nthreads);
    }
  }

  // F~_alpha = sum_i S[alpha][i] (f^inv_i(U) - f^visc_i(U, G)) for the n points of the chunk, in place over G's rows
  __device__ __forceinline__ void transform(const ChunkDesc &cd, long long, long long pl, T *stage, int LDB, int NE, int tid,
                                            int nthreads) const {
    const int n = cd.nrows;
    const int lgne = 31 - __clz(NE);
    const T *sm = stage + 4 * n * LDB;
    const int sstr = curved ? n * NE : NE;   // stride between the 9 metric components
    for (int p = tid; p < (n << lgne); p += nthreads) {
      const int j = p >> lgne, e = p - (j << lgne);
      T *col = stage + e;
      T uu[5];
#pragma unroll
      for (int v = 0; v < 5; ++v) uu[v] = col[(3 * n + j) * LDB + v * NE];
      T f[3][5], rr, vel[3], pr;
      inviscid_flux(uu, ph.gamma, f, rr, vel, pr);
      if (ph.ns) {
        T q[3][5];
#pragma unroll
        for (int i = 0; i < 3; ++i)
#pragma unroll
          for (int v = 0; v < 5; ++v) q[i][v] = col[(i * n + j) * LDB + v * NE];
        subtract_viscous_flux(uu, q, rr, vel, ph.gamma, ph.mu, ph.prandtl, f);
      }
      const T *sp = sm + (curved ? j * NE : 0) + e;
      const bool live = pl * NE + e < neles;
#pragma unroll
      for (int a = 0; a < 3; ++a) {
        const T s0 = sp[(a * 3 + 0) * sstr], s1 = sp[(a * 3 + 1) * sstr], s2 = sp[(a * 3 + 2) * sstr];
#pragma unroll
        for (int v = 0; v < 5; ++v) col[(a * n + j) * LDB + v * NE] = live ? s0 * f[0][v] + s1 * f[1][v] + s2 * f[2][v] : T(0);
      }
    }
  }
};

template <typename T, int EW>
struct VecIO;
template <>
struct VecIO<double, 2> {
  static __device__ __forceinline__ void ld(const double *p, double (&x)[2]) {
    const double2 t = *reinterpret_cast<const double2 *>(p);
    x[0] = t.x;
    x[1] = t.y;
  }
  static __device__ __forceinline__ void st(double *p, const double (&x)[2]) { *reinterpret_cast<double2 *>(p) = make_double2(x[0], x[1]); }
};
template <>
struct VecIO<float, 2> {
  static __device__ __forceinline__ void ld(const float *p, float (&x)[2]) {
    const float2 t = *reinterpret_cast<const float2 *>(p);
    x[0] = t.x;
    x[1] = t.y;
  }
  static __device__ __forceinline__ void st(float *p, const float (&x)[2]) { *reinterpret_cast<float2 *>(p) = make_float2(x[0], x[1]); }
};
template <>
struct VecIO<float, 1> {
  static __device__ __forceinline__ void ld(const float *p, float (&x)[1]) { x[0] = *p; }
  static __device__ __forceinline__ void st(float *p, const float (&x)[1]) { *p = x[0]; }
};

// K = -R/|J| (S9), then the stage update out1 = in1 + c1 K, out2 = in2 + c2 K (S10) or plain out1 = K
template <typename T>
struct RkEpilogue {
  const T *rcpdjac;
  long long ld, neles;
  int curved, NE;
  StageArgs<T> sa;
  template <typename ACC>
  __device__ __forceinline__ void operator()(ACC &acc, const int *rowmap, int slot0, long long, long long pl, int wc, int lane) const {
    constexpr int EW = ACC::EW;
    const long long e0 = pl * NE;
    T c1 = T(0), c2 = T(0);
    if (sa.coef) {
      c1 = (T)sa.coef->c1;
      c2 = (T)sa.coef->c2;
    }
    int mrow[ACC::NSLOT][ACC::ROWS];
    acc.foreach_row(lane, [&](int i, int rr, int r) { mrow[i][rr] = rowmap[(slot0 + i) * 8 + r]; });
    acc.foreach_tile(wc, lane, [&](int i, int rr, int e, T(&tile)[PV][EW]) {
      const int m = mrow[i][rr];
      if (m < 0) return;
      const long long col = e0 + e;
      T rj[EW];
      VecIO<T, EW>::ld(rcpdjac + (curved ? (long long)m * ld : 0) + col, rj);
      bool live[EW];
#pragma unroll
      for (int j = 0; j < EW; ++j) live[j] = col + j < neles;
#pragma unroll
      for (int v = 0; v < PV; ++v) {
        const long long idx = ((long long)m * 5 + v) * ld + col;
        T k[EW], o1[EW];
#pragma unroll
        for (int j = 0; j < EW; ++j) k[j] = live[j] ? -tile[v][j] * rj[j] : T(0);
        if (!sa.coef) {
          VecIO<T, EW>::st(sa.out1 + idx, k);
        } else {
          T a[EW];
          VecIO<T, EW>::ld(sa.in1 + idx, a);
          if (sa.out2) {
            T b[EW], o2[EW];
            VecIO<T, EW>::ld(sa.in2 + idx, b);
#pragma unroll
            for (int j = 0; j < EW; ++j) o2[j] = live[j] ? b[j] + c2 * k[j] : T(0);
            VecIO<T, EW>::st(sa.out2 + idx, o2);
          }
#pragma unroll
          for (int j = 0; j < EW; ++j) o1[j] = live[j] ? a[j] + c1 * k[j] : T(0);
          VecIO<T, EW>::st(sa.out1 + idx, o1);
        }
      }
    });
  }
};

template <typename T>
struct DivArgs {
  PanelOp<T> op;
  FluxProducer<T> prod;
  RkEpilogue<T> epi;
  long long npanels;
};

template <typename T, int NIT, int CX>
__global__ void __launch_bounds__(32 * panel_maxw<T>(NIT, CX)) k_fused_div(const __grid_constant__ DivArgs<T> a) {
  extern __shared__ __align__(16) char panel_smem[];
  panel_mainloop<T, NIT, CX>(a.op, a.prod, a.epi, a.npanels, 1, panel_smem);
}

// ------------------------------------------------------------------------------------------------ fused_grad
// epilogue S4: physical gradient from the three reference components held by one thread
template <typename T>
struct GradEpilogue {
  const T *smats, *rcpdjac;
  T *grad;                  // [3][Nu][5][ld]
  long long ld, neles;
  int nupts, curved, NE;
  template <typename ACC>
  __device__ __forceinline__ void operator()(ACC &acc, const int *rowmap, int slot0, long long, long long pl, int wc, int lane) const {
    constexpr int EW = ACC::EW;
    const long long e0 = pl * NE;
    int mrow[ACC::NSLOT][ACC::ROWS];
    acc.foreach_row(lane, [&](int i, int rr, int r) { mrow[i][rr] = rowmap[(slot0 + i) * 8 + r]; });
    acc.foreach_triple(wc, lane, [&](int t, int rr, int e, T(&t0)[PV][EW], T(&t1)[PV][EW], T(&t2)[PV][EW]) {
      const int rho = mrow[3 * t][rr];     // alpha = 0 rows are 0..Nu-1
      if (rho < 0) return;
      const long long col = e0 + e;
      T rj[EW], S[3][3][EW];
      VecIO<T, EW>::ld(rcpdjac + (curved ? (long long)rho * ld : 0) + col, rj);
#pragma unroll
      for (int a = 0; a < 3; ++a)
#pragma unroll
        for (int i = 0; i < 3; ++i)
          VecIO<T, EW>::ld(smats + (curved ? ((long long)(a * 3 + i) * nupts + rho) * ld : (long long)(a * 3 + i) * ld) + col, S[a][i]);
#pragma unroll
      for (int j = 0; j < EW; ++j)
        if (col + j >= neles) rj[j] = T(0);      // padding lanes: zero
#pragma unroll
      for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int v = 0; v < PV; ++v) {
          T o[EW];
#pragma unroll
          for (int j = 0; j < EW; ++j) o[j] = rj[j] * (S[0][i][j] * t0[v][j] + S[1][i][j] * t1[v][j] + S[2][i][j] * t2[v][j]);
          VecIO<T, EW>::st(grad + (((long long)i * nupts + rho) * 5 + v) * ld + col, o);
        }
    });
  }
};

template <typename T>
struct GradArgs {
  PanelOp<T> op;
  PlainProducer<T> prod;
  GradEpilogue<T> epi;
  long long npanels;
};

template <typename T, int NIT, int CX>
__global__ void __launch_bounds__(32 * panel_maxw<T>(NIT, CX)) k_fused_grad(const __grid_constant__ GradArgs<T> a) {
  extern __shared__ __align__(16) char panel_smem[];
  panel_mainloop<T, NIT, CX>(a.op, a.prod, a.epi, a.npanels, 1, panel_smem);
}

template <typename K, typename A>
void launch_panel(K k, const A &a, int nthreads, size_t smem, long long ntot, cudaStream_t s) {
  FR_CUDA_TRY(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  const long long grid = std::min<long long>(ntot, device_sm_count());
  k<<<(unsigned)grid, nthreads, smem, s>>>(a);
  FR_CUDA_TRY(cudaGetLastError());
}

}  // namespace

template <typename T>
bool fused_div_build(PanelOp<T> &op, int nu, int nf, const double *M132, const double *M3, int curved) {
  const int K = 3 * nu + nf;
  std::vector<double> A((size_t)nu * K);
  for (int m = 0; m < nu; ++m) {
    for (int k = 0; k < 3 * nu; ++k) A[(size_t)m * K + k] = M132[(size_t)m * 3 * nu + k];
    for (int k = 0; k < nf; ++k) A[(size_t)m * K + 3 * nu + k] = M3[(size_t)m * nf + k];
  }
  std::vector<KSource> srcs{KSource{nu, KIND_FLUX, 1}, KSource{nf, KIND_PLAIN, 1}};
  PackOptions opt;
  opt.min_ne = 16;
  opt.max_ne = 64;
  opt.curved = curved;
  return panel_op_build(op, nu, K, A.data(), srcs, opt, 150 * 1024);
}

template <typename T>
int launch_fused_div(const PanelOp<T> &op, const EleView<T> &ev, const T *u, const T *grad, const T *d, const PhysParams<T> &ph,
                     const StageArgs<T> &sa, cudaStream_t s) {
  DivArgs<T> a;
  a.op = op;
  a.prod = FluxProducer<T>{u, grad, d, ev.smats, ev.ld, ev.neles, ev.nupts, ev.affine ? 0 : 1, ph};
  a.epi = RkEpilogue<T>{ev.rcpdjac, ev.ld, ev.neles, ev.affine ? 0 : 1, op.NE, sa};
  a.npanels = ev.ld / op.NE;
  const size_t smem = panel_smem_bytes(op);
  const int nthreads = 32 * op.WR * op.WC;
#define FR_CASE(NIT_, CX_)                                                          \
  if (op.NIT == NIT_ && op.CX == CX_) {                                             \
    launch_panel(k_fused_div<T, NIT_, CX_>, a, nthreads, smem, a.npanels, s);       \
    return 1;                                                                       \
  }
  if constexpr (sizeof(T) == 8) {
    FR_PANEL_SHAPES_F64(FR_CASE)
  } else {
    FR_PANEL_SHAPES_F32(FR_CASE)
  }
#undef FR_CASE
  throw Error{FR_ESTATE, "launch_fused_div: no kernel for this accumulator shape"};
}

template <typename T>
bool fused_grad_build(PanelOp<T> &op, int nu, int nf, const double *M460, const double *M6) {
  const int K = nu + nf, M = 3 * nu;
  std::vector<double> A((size_t)M * K);
  for (int m = 0; m < M; ++m) {
    for (int k = 0; k < nu; ++k) A[(size_t)m * K + k] = M460[(size_t)m * nu + k];
    for (int k = 0; k < nf; ++k) A[(size_t)m * K + nu + k] = M6[(size_t)m * nf + k];
  }
  std::vector<KSource> srcs{KSource{nu, KIND_PLAIN, 1}, KSource{nf, KIND_PLAIN, 1}};
  PackOptions opt;
  opt.min_ne = 16;
  opt.max_ne = 64;
  opt.triple = 1;
  return panel_op_build(op, M, K, A.data(), srcs, opt, 150 * 1024);
}

template <typename T>
int launch_fused_grad(const PanelOp<T> &op, const EleView<T> &ev, const T *u, const T *c, T *grad, cudaStream_t s) {
  GradArgs<T> a;
  a.op = op;
  ColMap cm{op.NE, ev.ld, 0, ev.ld};
  a.prod.src[0] = MatRef<T>{u, 5 * ev.ld, 0};
  a.prod.src[1] = MatRef<T>{c, 5 * ev.ld, 0};
  a.prod.cm = cm;
  a.epi = GradEpilogue<T>{ev.smats, ev.rcpdjac, grad, ev.ld, ev.neles, ev.nupts, ev.affine ? 0 : 1, op.NE};
  a.npanels = ev.ld / op.NE;
  const size_t smem = panel_smem_bytes(op);
  const int nthreads = 32 * op.WR * op.WC;
#define FR_CASE(NIT_, CX_)                                                          \
  if (op.NIT == NIT_ && op.CX == CX_) {                                             \
    launch_panel(k_fused_grad<T, NIT_, CX_>, a, nthreads, smem, a.npanels, s);      \
    return 1;                                                                       \
  }
  if constexpr (sizeof(T) == 8) {
    FR_PANEL_TRIPLES_F64(FR_CASE)
  } else {
    FR_PANEL_TRIPLES_F32(FR_CASE)
  }
#undef FR_CASE
  throw Error{FR_ESTATE, "launch_fused_grad: no kernel for this accumulator shape"};
}

#define FR_INST(T)                                                                                                          \
  template bool fused_div_build<T>(PanelOp<T> &, int, int, const double *, const double *, int);                          \
  template int launch_fused_div<T>(const PanelOp<T> &, const EleView<T> &, const T *, const T *, const T *,                \
                                   const PhysParams<T> &, const StageArgs<T> &, cudaStream_t);                             \
  template bool fused_grad_build<T>(PanelOp<T> &, int, int, const double *, const double *);                               \
  template int launch_fused_grad<T>(const PanelOp<T> &, const EleView<T> &, const T *, const T *, T *, cudaStream_t);
FR_INST(double)
FR_INST(float)

}  // namespace frb
