// Fused panel kernels (fusion targets F-A and F-B of SURVEY 7.2):
//   fused_grad: S3 + S4              G_i = (1/|J|) sum_alpha S[alpha][i] ( [M460 | M6] [U; C] )_alpha
//               the three alpha components of a solution point sit in one thread (triple packing), so the transform to
//               physical gradients is formed in registers in the epilogue;
//   fused_div : S8 + S9 + S10        dudt = -(1/|J|) [ M132 | M3 ] [F~; D]  (+ Runge-Kutta stage update in the epilogue).
// (A first version formed F~ inside fused_div from U, G and the metrics staged in shared memory; ncu showed the CTA waiting
//  at barriers on a long, serial FP64 flux evaluation that only part of the threads could share, profiles/r01_*.md.)
// Both run on the persistent panel main loop (panel_kernel.cuh) with the operator resident in shared memory.
#include "kernels.cuh"
#include "panel_kernel.cuh"

namespace frb {

namespace {

// ------------------------------------------------------------------------------------------------ fused_div
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
  // read-only data (metrics): ld.global.nc tells the compiler the load cannot alias the epilogue's stores, so the loads of the
  // next tile may be hoisted above the stores of this one
  static __device__ __forceinline__ void ldg(const double *p, double (&x)[2]) {
    const double2 t = __ldg(reinterpret_cast<const double2 *>(p));
    x[0] = t.x;
    x[1] = t.y;
  }
};
template <>
struct VecIO<float, 2> {
  static __device__ __forceinline__ void ld(const float *p, float (&x)[2]) {
    const float2 t = *reinterpret_cast<const float2 *>(p);
    x[0] = t.x;
    x[1] = t.y;
  }
  static __device__ __forceinline__ void st(float *p, const float (&x)[2]) { *reinterpret_cast<float2 *>(p) = make_float2(x[0], x[1]); }
  static __device__ __forceinline__ void ldg(const float *p, float (&x)[2]) {
    const float2 t = __ldg(reinterpret_cast<const float2 *>(p));
    x[0] = t.x;
    x[1] = t.y;
  }
};
template <>
struct VecIO<float, 1> {
  static __device__ __forceinline__ void ld(const float *p, float (&x)[1]) { x[0] = *p; }
  static __device__ __forceinline__ void st(float *p, const float (&x)[1]) { *p = x[0]; }
  static __device__ __forceinline__ void ldg(const float *p, float (&x)[1]) { x[0] = __ldg(p); }
};

// K = -R/|J| (S9), then the stage update out1 = in1 + c1 K, out2 = in2 + c2 K (S10) or plain out1 = K
template <typename T>
struct RkEpilogue {
  const T *rcpdjac;
  long long ld, neles;
  int curved, NE;
  StageArgs<T> sa;
  template <typename ACC>
  __device__ __forceinline__ void prefetch(ACC &acc, const int *rowmap, int slot0, long long, long long pl, int wc, int lane) const {
    const long long e0 = pl * NE;
    acc.foreach_coord(wc, lane, [&](int i, int rr, int e) {
      const int m = rowmap[(slot0 + i) * 8 + (ACC::ROWS == 1 ? (lane >> 2) : rr)];
      if (m < 0) return;
      const long long col = e0 + e;
      if (curved || i == 0) prefetch_l2(rcpdjac + (curved ? (long long)m * ld : 0) + col);
      if (!sa.coef) return;
#pragma unroll
      for (int v = 0; v < PV; ++v) {
        const long long idx = ((long long)m * 5 + v) * ld + col;
        prefetch_l2(sa.in1 + idx);
        if (sa.out2 && sa.in2 != sa.in1) prefetch_l2(sa.in2 + idx);
      }
    });
  }
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
    const bool same = sa.in2 == sa.in1;
    acc.foreach_tile(wc, lane, [&](int i, int rr, int e, T(&tile)[PV][EW]) {
      const int m = mrow[i][rr];
      if (m < 0) return;
      const long long col = e0 + e;
      const long long idx0 = (long long)m * 5 * ld + col;
      T rj[EW];
      VecIO<T, EW>::ldg(rcpdjac + (curved ? (long long)m * ld : 0) + col, rj);
      bool live[EW];
#pragma unroll
      for (int j = 0; j < EW; ++j) live[j] = col + j < neles;
      if constexpr (sizeof(T) == 4) {
        // FP32: all global loads of the tile first -- the stores below may alias them, so the compiler would otherwise
        // serialise load -> store -> load and expose one memory latency per variable.  (In FP64 the 20 extra registers
        // spill: 0.95 -> 1.57 ms on the tetrahedra, so FP64 keeps the load-per-variable order.)
        T a[PV][EW], b[PV][EW];
        if (sa.coef) {
#pragma unroll
          for (int v = 0; v < PV; ++v) VecIO<T, EW>::ld(sa.in1 + idx0 + v * ld, a[v]);
          if (sa.out2 && !same) {
#pragma unroll
            for (int v = 0; v < PV; ++v) VecIO<T, EW>::ld(sa.in2 + idx0 + v * ld, b[v]);
          }
        }
#pragma unroll
        for (int v = 0; v < PV; ++v) {
          const long long idx = idx0 + v * ld;
          T k[EW], o1[EW];
#pragma unroll
          for (int j = 0; j < EW; ++j) k[j] = live[j] ? -tile[v][j] * rj[j] : T(0);
          if (!sa.coef) {
            VecIO<T, EW>::st(sa.out1 + idx, k);
          } else {
            if (sa.out2) {
              T o2[EW];
#pragma unroll
              for (int j = 0; j < EW; ++j) o2[j] = live[j] ? (same ? a[v][j] : b[v][j]) + c2 * k[j] : T(0);
              VecIO<T, EW>::st(sa.out2 + idx, o2);
            }
#pragma unroll
            for (int j = 0; j < EW; ++j) o1[j] = live[j] ? a[v][j] + c1 * k[j] : T(0);
            VecIO<T, EW>::st(sa.out1 + idx, o1);
          }
        }
      } else if (sa.coef && same) {
        // FP64, RK45[2R+] (both updates start from the same register X): the five loads of the tile together, then the stores
        T a[PV][EW];
#pragma unroll
        for (int v = 0; v < PV; ++v) VecIO<T, EW>::ld(sa.in1 + idx0 + v * ld, a[v]);
#pragma unroll
        for (int v = 0; v < PV; ++v) {
          const long long idx = idx0 + v * ld;
          T k[EW], o1[EW];
#pragma unroll
          for (int j = 0; j < EW; ++j) k[j] = live[j] ? -tile[v][j] * rj[j] : T(0);
          if (sa.out2) {
            T o2[EW];
#pragma unroll
            for (int j = 0; j < EW; ++j) o2[j] = live[j] ? a[v][j] + c2 * k[j] : T(0);
            VecIO<T, EW>::st(sa.out2 + idx, o2);
          }
#pragma unroll
          for (int j = 0; j < EW; ++j) o1[j] = live[j] ? a[v][j] + c1 * k[j] : T(0);
          VecIO<T, EW>::st(sa.out1 + idx, o1);
        }
      } else {
#pragma unroll
        for (int v = 0; v < PV; ++v) {
          const long long idx = idx0 + v * ld;
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
              if (!same) {
                VecIO<T, EW>::ld(sa.in2 + idx, b);
              } else {
#pragma unroll
                for (int j = 0; j < EW; ++j) b[j] = a[j];
              }
#pragma unroll
              for (int j = 0; j < EW; ++j) o2[j] = live[j] ? b[j] + c2 * k[j] : T(0);
              VecIO<T, EW>::st(sa.out2 + idx, o2);
            }
#pragma unroll
            for (int j = 0; j < EW; ++j) o1[j] = live[j] ? a[j] + c1 * k[j] : T(0);
            VecIO<T, EW>::st(sa.out1 + idx, o1);
          }
        }
      }
    });
  }
};

template <typename T>
struct alignas(64) DivArgs {
  TmaProducer<T> prod;
  PanelOp<T> op;
  RkEpilogue<T> epi;
  long long npanels;
};

template <typename T, int NIT, int CX>
__global__ void __launch_bounds__(32 * panel_maxw<T>(NIT, CX)) k_fused_div(const __grid_constant__ DivArgs<T> a) {
  extern __shared__ __align__(1024) char panel_smem[];
  panel_mainloop<T, NIT, CX>(a.op, a.prod, a.epi, a.npanels, 1, panel_smem);
}

// ------------------------------------------------------------------------------------------------ fused_grad
// epilogue S4: physical gradient from the three reference components held by one thread
template <typename T>
struct GradEpilogue {
  const T *smats, *rcpdjac;
  T *grad;                  // [3][Nu][5][ld]  physical gradients G (read again by S5 and S6)
  long long ld, neles;
  int nupts, curved, NE;
  template <typename ACC>
  __device__ __forceinline__ void prefetch(ACC &acc, const int *rowmap, int slot0, long long, long long pl, int wc, int lane) const {
    const long long e0 = pl * NE;
    if (!curved && slot0 != 0) return;      // per-element metric terms: the first row-warp's prefetch covers the panel
    acc.foreach_coord(wc, lane, [&](int i, int rr, int e) {
      if (i % 3 != 0) return;
      const int rho = rowmap[(slot0 + i) * 8 + (ACC::ROWS == 1 ? (lane >> 2) : rr)];
      if (rho < 0 || (!curved && i != 0)) return;
      const long long col = e0 + e;
      prefetch_l2(rcpdjac + (curved ? (long long)rho * ld : 0) + col);
#pragma unroll
      for (int a = 0; a < 9; ++a) prefetch_l2(smats + (curved ? ((long long)a * nupts + rho) * ld : (long long)a * ld) + col);
    });
  }
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
      VecIO<T, EW>::ldg(rcpdjac + (curved ? (long long)rho * ld : 0) + col, rj);
#pragma unroll
      for (int a = 0; a < 3; ++a)
#pragma unroll
        for (int i = 0; i < 3; ++i)
          VecIO<T, EW>::ldg(smats + (curved ? ((long long)(a * 3 + i) * nupts + rho) * ld : (long long)(a * 3 + i) * ld) + col, S[a][i]);
#pragma unroll
      for (int j = 0; j < EW; ++j)
        if (col + j >= neles) rj[j] = T(0);      // padding lanes: zero
#pragma unroll
      for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int v = 0; v < PV; ++v) {
          T q[EW];
#pragma unroll
          for (int j = 0; j < EW; ++j) q[j] = rj[j] * (S[0][i][j] * t0[v][j] + S[1][i][j] * t1[v][j] + S[2][i][j] * t2[v][j]);
          VecIO<T, EW>::st(grad + (((long long)i * nupts + rho) * 5 + v) * ld + col, q);
        }
    });
  }
};

template <typename T>
struct alignas(64) GradArgs {
  TmaProducer<T> prod;
  PanelOp<T> op;
  GradEpilogue<T> epi;
  long long npanels;
};

template <typename T, int NIT, int CX>
__global__ void __launch_bounds__(32 * panel_maxw<T>(NIT, CX)) k_fused_grad(const __grid_constant__ GradArgs<T> a) {
  extern __shared__ __align__(1024) char panel_smem[];
  panel_mainloop<T, NIT, CX>(a.op, a.prod, a.epi, a.npanels, 1, panel_smem);
}

}  // namespace

template <typename T>
bool fused_div_build(PanelOp<T> &op, int nu, int nf, const double *M132, const double *M3, int cand, int r0, int nr) {
  // rows r0 .. r0+nr-1 of [M132 | M3] (nr < 0: all); the epilogue sees the solution-point numbers through the row map
  if (nr < 0) {
    r0 = 0;
    nr = nu;
  }
  const int K = 3 * nu + nf;
  std::vector<double> A((size_t)nr * K);
  std::vector<int> ids(nr);
  for (int j = 0; j < nr; ++j) {
    const int m = r0 + j;
    ids[j] = m;
    for (int k = 0; k < 3 * nu; ++k) A[(size_t)j * K + k] = M132[(size_t)m * 3 * nu + k];
    for (int k = 0; k < nf; ++k) A[(size_t)j * K + 3 * nu + k] = M3[(size_t)m * nf + k];
  }
  std::vector<KSource> srcs{KSource{3 * nu}, KSource{nf}};
  PackOptions opt;
  opt.min_ne = sizeof(T) == 8 ? 16 : 32;
  opt.max_ne = sizeof(T) == 8 ? 64 : 128;
  opt.cand = cand;
  opt.row_ids = ids.data();
  return panel_op_build(op, nr, K, A.data(), srcs, opt, 150 * 1024);
}

template <typename T>
int launch_fused_div(const PanelOp<T> &op, const EleView<T> &ev, const T *ftil, const T *d, const StageArgs<T> &sa,
                     cudaStream_t s) {
  DivArgs<T> a;
  a.op = op;
  a.op.pf_epi = 1;
  a.prod.tm[0] = tmap_state(ftil, 3ll * ev.nupts, ev.ld, op.NE, op.src_step[0]);
  a.prod.tm[1] = tmap_state(d, (long long)ev.nfpts, ev.ld, op.NE, op.src_step[1]);
  a.prod.plain = 0;
  a.epi = RkEpilogue<T>{ev.rcpdjac, ev.ld, ev.neles, ev.affine ? 0 : 1, op.NE, sa};
  a.npanels = ev.ld / op.NE;
#define FR_CASE(NIT_, CX_)                                                          \
  if (op.NIT == NIT_ && op.CX == CX_) {                                             \
    panel_launch(k_fused_div<T, NIT_, CX_>, a, op, a.npanels, s);                   \
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
bool fused_grad_build(PanelOp<T> &op, int nu, int nf, const double *M460, const double *M6, int cand, const double *M0_jump,
                      int r0, int nr) {
  // rows (alpha, rho), rho = r0 .. r0+nr-1, of [M460 | M6] (nr < 0: all rho), alpha-major as triple packing wants them
  if (nr < 0) {
    r0 = 0;
    nr = nu;
  }
  const int K = nu + nf, M = 3 * nr;
  std::vector<double> A((size_t)M * K);
  std::vector<int> ids(M);
  for (int a = 0; a < 3; ++a)
    for (int j = 0; j < nr; ++j) {
      const int ml = a * nr + j, m = a * nu + r0 + j;
      ids[ml] = m;
      for (int k = 0; k < nu; ++k) A[(size_t)ml * K + k] = M460[(size_t)m * nu + k];
      for (int k = 0; k < nf; ++k) A[(size_t)ml * K + nu + k] = M6[(size_t)m * nf + k];
      // jump formulation (k_con_u): the second operand is C - U_f, so the first block is M4 = M460 + M6 M0
      if (M0_jump)
        for (int k = 0; k < nu; ++k) {
          double acc = 0;
          for (int i = 0; i < nf; ++i) acc += M6[(size_t)m * nf + i] * M0_jump[(size_t)i * nu + k];
          A[(size_t)ml * K + k] += acc;
        }
    }
  std::vector<KSource> srcs{KSource{nu}, KSource{nf}};
  PackOptions opt;
  opt.min_ne = sizeof(T) == 8 ? 16 : 32;
  opt.max_ne = sizeof(T) == 8 ? 64 : 128;
  opt.triple = 1;
  opt.cand = cand;
  opt.row_ids = ids.data();
  return panel_op_build(op, M, K, A.data(), srcs, opt, 150 * 1024);
}

template <typename T>
int launch_fused_grad(const PanelOp<T> &op, const EleView<T> &ev, const T *u, const T *c, T *grad, cudaStream_t s) {
  GradArgs<T> a;
  a.op = op;
  // The L2 prefetch of the epilogue's metric terms pays only in FP64 with per-element terms; with per-point terms (20 lines per
  // thread) and in FP32 it costs more issue slots than the latency it hides (profiles/r01_j_panel_source_level.md item 7).
  a.op.pf_epi = (ev.affine && sizeof(T) == 8) ? 1 : 0;
  a.prod.tm[0] = tmap_state(u, (long long)ev.nupts, ev.ld, op.NE, op.src_step[0]);
  a.prod.tm[1] = tmap_state(c, (long long)ev.nfpts, ev.ld, op.NE, op.src_step[1]);
  a.prod.plain = 0;
  a.epi = GradEpilogue<T>{ev.smats, ev.rcpdjac, grad, ev.ld, ev.neles, ev.nupts, ev.affine ? 0 : 1, op.NE};
  a.npanels = ev.ld / op.NE;
#define FR_CASE(NIT_, CX_)                                                          \
  if (op.NIT == NIT_ && op.CX == CX_) {                                             \
    panel_launch(k_fused_grad<T, NIT_, CX_>, a, op, a.npanels, s);                  \
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
  template bool fused_div_build<T>(PanelOp<T> &, int, int, const double *, const double *, int, int, int);                             \
  template int launch_fused_div<T>(const PanelOp<T> &, const EleView<T> &, const T *, const T *, const StageArgs<T> &,     \
                                   cudaStream_t);                                                                          \
  template bool fused_grad_build<T>(PanelOp<T> &, int, int, const double *, const double *, int, const double *, int, int);                             \
  template int launch_fused_grad<T>(const PanelOp<T> &, const EleView<T> &, const T *, const T *, T *, cudaStream_t);
FR_INST(double)
FR_INST(float)

}  // namespace frb
