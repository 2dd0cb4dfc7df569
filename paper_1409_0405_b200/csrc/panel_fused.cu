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
  static constexpr bool kProducerPrefetch = false;
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
      const T *p1 = sa.in1 + (long long)m * 5 * ld + col, *p2 = sa.in2 + (long long)m * 5 * ld + col;
#pragma unroll
      for (int v = 0; v < PV; ++v) {
        prefetch_l2(p1);
        if (sa.out2 && sa.in2 != sa.in1) prefetch_l2(p2);
        p1 += ld;
        p2 += ld;
      }
    });
  }
  // One tile (row m, EW consecutive elements, all variables).  MASK: the panel holds padding columns (col >= neles), which are
  // written as zero whatever the accumulators hold; interior panels skip the selects.
  template <bool MASK, int EW>
  __device__ __forceinline__ void tile_update(T (&tile)[PV][EW], int m, long long col, T c1, T c2, bool same) const {
    const long long idx0 = (long long)m * 5 * ld + col;
    T rj[EW];
    VecIO<T, EW>::ldg(rcpdjac + (curved ? (long long)m * ld : 0) + col, rj);
    bool live[EW];
#pragma unroll
    for (int j = 0; j < EW; ++j) live[j] = !MASK || col + j < neles;
    auto sel = [&](int j, T x) { return (!MASK || live[j]) ? x : T(0); };
    if (!sa.coef) {
      T *o = sa.out1 + idx0;
#pragma unroll
      for (int v = 0; v < PV; ++v) {
        T k[EW];
#pragma unroll
        for (int j = 0; j < EW; ++j) k[j] = sel(j, -tile[v][j] * rj[j]);
        VecIO<T, EW>::st(o, k);
        o += ld;
      }
      return;
    }
    // the loads of the tile together, then the stores: the stores may alias the loads, so the compiler would otherwise serialise
    // load -> store -> load and expose one memory latency per variable
    T a[PV][EW];
    const T *pa = sa.in1 + idx0;
#pragma unroll
    for (int v = 0; v < PV; ++v) {
      VecIO<T, EW>::ld(pa, a[v]);
      pa += ld;
    }
    T *o1p = sa.out1 + idx0, *o2p = sa.out2 + idx0;
    if (sa.out2 && !same) {
      const T *pb = sa.in2 + idx0;
#pragma unroll
      for (int v = 0; v < PV; ++v) {
        T bb[EW], k[EW], o1[EW], o2[EW];
        VecIO<T, EW>::ld(pb, bb);
#pragma unroll
        for (int j = 0; j < EW; ++j) {
          k[j] = -tile[v][j] * rj[j];
          o2[j] = sel(j, bb[j] + c2 * k[j]);
          o1[j] = sel(j, a[v][j] + c1 * k[j]);
        }
        VecIO<T, EW>::st(o2p, o2);
        VecIO<T, EW>::st(o1p, o1);
        pb += ld;
        o1p += ld;
        o2p += ld;
      }
      return;
    }
#pragma unroll
    for (int v = 0; v < PV; ++v) {
      T k[EW], o1[EW];
#pragma unroll
      for (int j = 0; j < EW; ++j) k[j] = -tile[v][j] * rj[j];
      if (sa.out2) {
        T o2[EW];
#pragma unroll
        for (int j = 0; j < EW; ++j) o2[j] = sel(j, a[v][j] + c2 * k[j]);
        VecIO<T, EW>::st(o2p, o2);
        o2p += ld;
      }
#pragma unroll
      for (int j = 0; j < EW; ++j) o1[j] = sel(j, a[v][j] + c1 * k[j]);
      VecIO<T, EW>::st(o1p, o1);
      o1p += ld;
    }
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
    if (e0 + NE <= neles) {
      acc.foreach_tile(wc, lane, [&](int i, int rr, int e, T(&tile)[PV][EW]) {
        if (mrow[i][rr] >= 0) tile_update<false, EW>(tile, mrow[i][rr], e0 + e, c1, c2, same);
      });
    } else {
      acc.foreach_tile(wc, lane, [&](int i, int rr, int e, T(&tile)[PV][EW]) {
        if (mrow[i][rr] >= 0) tile_update<true, EW>(tile, mrow[i][rr], e0 + e, c1, c2, same);
      });
    }
  }
};

template <typename T>
struct alignas(64) DivArgs {
  TmaProducer<T> prod;
  PanelOp<T> op;
  RkEpilogue<T> epi;
  long long npanels;
};

template <typename T, int NIT, int CX, bool DYN>
__global__ void __launch_bounds__(32 * panel_maxw<T>(NIT, CX)) k_fused_div(const __grid_constant__ DivArgs<T> a) {
  extern __shared__ __align__(1024) char panel_smem[];
  panel_mainloop<T, NIT, CX, TmaProducer<T>, RkEpilogue<T>, true, false, DYN>(a.op, a.prod, a.epi, a.npanels, 1, panel_smem);
}

// ------------------------------------------------------------------------------------------------ fused_grad
// epilogue S4: physical gradient from the three reference components held by one thread
// PF: per-point metric terms (curved / non-affine types) prefetched into L2 by the producer warp; a compile-time variant, so that
// the kernels of affine types stay as they are
struct EpiNoMaps {};
struct EpiMetricMaps {
  CUtensorMap tm_s, tm_j;   // smats [9][nupts][ld], rcpdjac [1][nupts][ld], boxes of one panel
};
template <typename T, bool PF>
struct GradEpilogue : std::conditional_t<PF, EpiMetricMaps, EpiNoMaps> {
  const T *smats, *rcpdjac;
  T *grad;                  // [3][Nu][5][ld]  physical gradients G (read again by S5 and S6)
  long long ld, neles;
  int nupts, curved, NE;
  // PF: the panel's metric terms through the maps, one instruction per array and panel, so that the epilogue's loads are L2 hits
  // without costing the consumer warps anything
  static constexpr bool kProducerPrefetch = PF;
  __device__ __forceinline__ void producer_prefetch(long long pl) const {
    if constexpr (PF) {
      tma_prefetch_3d(&this->tm_s, (int)(pl * NE), 0, 0);
      tma_prefetch_3d(&this->tm_j, (int)(pl * NE), 0, 0);
    }
  }
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
      const T *sp = smats + (curved ? (long long)rho * ld : 0) + col;
      const long long sstep = curved ? (long long)nupts * ld : ld;
#pragma unroll
      for (int a = 0; a < 9; ++a) {
        prefetch_l2(sp);
        sp += sstep;
      }
    });
  }
  // One solution point rho, EW consecutive elements: G_i = (1/|J|) sum_alpha S[alpha][i] G~_alpha, one column i of S at a time
  // (three metric loads live instead of nine).  Metric terms are stored [alpha*3 + i][point][ld].
  template <bool MASK, int EW>
  __device__ __forceinline__ void point_transform(T (&t0)[PV][EW], T (&t1)[PV][EW], T (&t2)[PV][EW], int rho, long long col) const {
    T rj[EW];
    VecIO<T, EW>::ldg(rcpdjac + (curved ? (long long)rho * ld : 0) + col, rj);
    if (MASK) {
#pragma unroll
      for (int j = 0; j < EW; ++j)
        if (col + j >= neles) rj[j] = T(0);
    }
    const long long sstep = curved ? (long long)nupts * ld : ld;      // between metric terms
    const T *sp = smats + (curved ? (long long)rho * ld : 0) + col;   // S[0][0]
    T *gp = grad + (long long)rho * 5 * ld + col;
    const long long gstep = (long long)nupts * 5 * ld;                 // between gradient components
#pragma unroll
    for (int i = 0; i < 3; ++i) {
      T s0[EW], s1[EW], s2[EW];
      VecIO<T, EW>::ldg(sp + i * sstep, s0);
      VecIO<T, EW>::ldg(sp + (3 + i) * sstep, s1);
      VecIO<T, EW>::ldg(sp + (6 + i) * sstep, s2);
#pragma unroll
      for (int j = 0; j < EW; ++j) {
        s0[j] *= rj[j];
        s1[j] *= rj[j];
        s2[j] *= rj[j];
      }
      T *o = gp;
#pragma unroll
      for (int v = 0; v < PV; ++v) {
        T q[EW];
#pragma unroll
        for (int j = 0; j < EW; ++j) {
          q[j] = s0[j] * t0[v][j] + s1[j] * t1[v][j] + s2[j] * t2[v][j];
          if (MASK && col + j >= neles) q[j] = T(0);     // 0 * (non-finite garbage of a padding column) would not be 0
        }
        VecIO<T, EW>::st(o, q);
        o += ld;
      }
      gp += gstep;
    }
  }
  template <typename ACC>
  __device__ __forceinline__ void operator()(ACC &acc, const int *rowmap, int slot0, long long, long long pl, int wc, int lane) const {
    constexpr int EW = ACC::EW;
    const long long e0 = pl * NE;
    int mrow[ACC::NSLOT][ACC::ROWS];
    acc.foreach_row(lane, [&](int i, int rr, int r) { mrow[i][rr] = rowmap[(slot0 + i) * 8 + r]; });
    if (e0 + NE <= neles) {
      acc.foreach_triple(wc, lane, [&](int t, int rr, int e, T(&t0)[PV][EW], T(&t1)[PV][EW], T(&t2)[PV][EW]) {
        const int rho = mrow[3 * t][rr];     // alpha = 0 rows are 0..Nu-1
        if (rho >= 0) point_transform<false, EW>(t0, t1, t2, rho, e0 + e);
      });
    } else {
      acc.foreach_triple(wc, lane, [&](int t, int rr, int e, T(&t0)[PV][EW], T(&t1)[PV][EW], T(&t2)[PV][EW]) {
        const int rho = mrow[3 * t][rr];
        if (rho >= 0) point_transform<true, EW>(t0, t1, t2, rho, e0 + e);
      });
    }
  }
};

template <typename T, bool PF>
struct alignas(64) GradArgs {
  TmaProducer<T> prod;
  PanelOp<T> op;
  GradEpilogue<T, PF> epi;
  long long npanels;
};

template <typename T, int NIT, int CX, bool PF, bool DYN>
__global__ void __launch_bounds__(32 * panel_maxw<T>(NIT, CX, true)) k_fused_grad(const __grid_constant__ GradArgs<T, PF> a) {
  extern __shared__ __align__(1024) char panel_smem[];
  // FP32: the scalar accumulator form (panel.cuh: the packed pairs do not fit this kernel's register budget)
  panel_mainloop<T, NIT, CX, TmaProducer<T>, GradEpilogue<T, PF>, false, false, DYN>(a.op, a.prod, a.epi, a.npanels, 1, panel_smem);
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
    if (panel_use_units(op)) panel_launch(k_fused_div<T, NIT_, CX_, true>, a, op, a.npanels, s); \
    else panel_launch(k_fused_div<T, NIT_, CX_, false>, a, op, a.npanels, s);       \
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

namespace {
template <typename T, bool PF>
int launch_fused_grad_pf(const PanelOp<T> &op, const EleView<T> &ev, const T *u, const T *c, T *grad, cudaStream_t s) {
  GradArgs<T, PF> a;
  a.op = op;
  // Affine types and FP32: the consumers pull the epilogue's metric terms into L2 while the panel's first chunk is multiplied; with
  // per-point terms in FP64 (20 lines per thread) that costs more than the latency it hides (pri S3+S4 0.94 -> 1.04 ms).  PF: the
  // producer warp prefetches them instead, and the consumers issue nothing.
  a.op.pf_epi = PF ? 0 : ((ev.affine || sizeof(T) == 4) ? 1 : 0);
  a.prod.tm[0] = tmap_state(u, (long long)ev.nupts, ev.ld, op.NE, op.src_step[0]);
  a.prod.tm[1] = tmap_state(c, (long long)ev.nfpts, ev.ld, op.NE, op.src_step[1]);
  a.prod.plain = 0;
  a.epi.smats = ev.smats;
  a.epi.rcpdjac = ev.rcpdjac;
  a.epi.grad = grad;
  a.epi.ld = ev.ld;
  a.epi.neles = ev.neles;
  a.epi.nupts = ev.nupts;
  a.epi.curved = ev.affine ? 0 : 1;
  a.epi.NE = op.NE;
  if constexpr (PF) {
    bool ok1 = false, ok2 = false;
    a.epi.tm_s = tmap_epi(ev.smats, 9, (long long)ev.nupts, ev.ld, op.NE, ok1);
    a.epi.tm_j = tmap_epi(ev.rcpdjac, 1, (long long)ev.nupts, ev.ld, op.NE, ok2);
    FR_REQUIRE(ok1 && ok2, "launch_fused_grad: metric maps");
  }
  a.npanels = ev.ld / op.NE;
#define FR_CASE(NIT_, CX_)                                                          \
  if (op.NIT == NIT_ && op.CX == CX_) {                                             \
    if (panel_use_units(op)) panel_launch(k_fused_grad<T, NIT_, CX_, PF, true>, a, op, a.npanels, s); \
    else panel_launch(k_fused_grad<T, NIT_, CX_, PF, false>, a, op, a.npanels, s);  \
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
}  // namespace

template <typename T>
int launch_fused_grad(const PanelOp<T> &op, const EleView<T> &ev, const T *u, const T *c, T *grad, cudaStream_t s) {
  // per-point metric terms within the box limits of a tensor map (256 rows): producer-side prefetch
  if (!ev.affine && ev.nupts <= 256) return launch_fused_grad_pf<T, true>(op, ev, u, c, grad, s);
  return launch_fused_grad_pf<T, false>(op, ev, u, c, grad, s);
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
