// The persistent panel main loop shared by the plain operator product and its fused variants (see panel.cuh).
#pragma once
#include "panel.cuh"

namespace frb {


// Where a panel's columns live in a global matrix: column(v, e) = p*pstride + v*vstride + e, valid iff
// p*pstride + v*vlim + e < lim.  State matrices [rows][5][ld]: pstride = NE, vstride = ld, vlim = 0, lim = ld.
// Plain matrices [rows][N] (fr_gemm): pstride = 5*NE, vstride = vlim = NE, lim = N.
struct ColMap {
  long long pstride, vstride, vlim, lim;
};

template <typename T>
struct MatRef {
  const T *p;
  long long ld, bstride;   // row stride, batch stride (elements)
};

// ---- producer: B chunks are plain rows of up to two stacked global matrices
template <typename T>
struct PlainProducer {
  MatRef<T> src[2];
  ColMap cm;
  static constexpr bool kTransform = false;
  // per-thread copy lane, fixed for the life of the CTA (init): each thread owns one 16-byte column piece (variable v,
  // elements e..e+CTV) and walks down the rows, so a piece costs two pointer bumps and the copy
  int l_sub, l_rpi, l_v, l_e, l_wide;
  __device__ __forceinline__ void init(int NE, int tid, int nthreads) {
    constexpr int CTV = 16 / (int)sizeof(T);
    const int lg = 31 - __clz(NE / CTV);
    const int ppr = PV << lg;                         // pieces per row
    l_wide = nthreads >= ppr;                         // the usual case: one sweep of the group covers >= 1 whole row
    l_rpi = l_wide ? nthreads / ppr : 1;              // rows per sweep
    l_sub = l_wide ? tid / ppr : 0;
    const int col = tid - l_sub * ppr;
    l_v = col >> lg;
    l_e = (col - (l_v << lg)) * CTV;
  }
  __device__ __forceinline__ void issue_col(const ChunkDesc &cd, long long batch, long long pl, T *stage, int LDB, int NE, int v,
                                            int e) const {
    constexpr int CTV = 16 / (int)sizeof(T);
    long long nv = cm.lim - pl * cm.pstride - v * cm.vlim - e;
    nv = nv < 0 ? 0 : (nv > CTV ? CTV : nv);
    const int nbytes = (int)nv * (int)sizeof(T);
    const T *mp = cd.src ? src[1].p : src[0].p;
    const long long mld = cd.src ? src[1].ld : src[0].ld, mbs = cd.src ? src[1].bstride : src[0].bstride;
    const T *g = mp;
    long long gstep = 0;
    if (nv > 0) {
      g = mp + batch * mbs + (long long)(cd.row0 + l_sub) * mld + pl * cm.pstride + v * cm.vstride + e;
      gstep = (long long)l_rpi * mld;
    }
    T *sp = stage + l_sub * LDB + v * NE + e;
    const int sstep = l_rpi * LDB;
    for (int r = l_sub; r < cd.nrows; r += l_rpi) {
      pcp_async16(sp, g, nbytes);
      g += gstep;
      sp += sstep;
    }
  }
  __device__ __forceinline__ void issue(const ChunkDesc &cd, long long batch, long long pl, T *stage, int LDB, int NE, int tid,
                                        int nthreads) const {
    if (l_wide) {
      if (l_sub < l_rpi) issue_col(cd, batch, pl, stage, LDB, NE, l_v, l_e);
      return;
    }
    constexpr int CTV = 16 / (int)sizeof(T);
    const int lg = 31 - __clz(NE / CTV);
    for (int col = tid; col < (PV << lg); col += nthreads) {
      const int v = col >> lg;
      issue_col(cd, batch, pl, stage, LDB, NE, v, (col - (v << lg)) * CTV);
    }
  }
  __device__ __forceinline__ void transform(const ChunkDesc &, long long, long long, T *, int, int, int, int) const {}
};

// ---- epilogue: C <- c1*acc + c2*C
template <typename T>
struct PlainEpilogue {
  T *C;
  long long ldc, bstride;
  ColMap cm;
  T c1, c2;
  template <typename ACC>
  __device__ __forceinline__ void prefetch(ACC &acc, const int *rowmap, int slot0, long long batch, long long pl, int wc,
                                           int lane) const {
    if (c2 == T(0)) return;
    const T *Cb = C + batch * bstride + pl * cm.pstride;
    acc.foreach_coord(wc, lane, [&](int i, int rr, int e) {
      const int m = rowmap[(slot0 + i) * 8 + (ACC::ROWS == 1 ? (lane >> 2) : rr)];
      if (m < 0) return;
#pragma unroll
      for (int v = 0; v < PV; ++v)
        if (pl * cm.pstride + v * cm.vlim + e < cm.lim) prefetch_l2(Cb + (long long)m * ldc + v * cm.vstride + e);
    });
  }
  template <typename ACC>
  __device__ __forceinline__ void operator()(ACC &acc, const int *rowmap, int slot0, long long batch, long long pl, int wc,
                                             int lane) const {
    T *Cb = C + batch * bstride + pl * cm.pstride;
    const long long vb = pl * cm.pstride;
    constexpr int EW = ACC::EW;
    const bool interior = vb + (PV - 1) * cm.vlim + (cm.pstride > cm.vstride ? cm.vstride : cm.pstride) <= cm.lim;
    int mrow[ACC::NSLOT][ACC::ROWS];
    acc.foreach_row(lane, [&](int i, int rr, int r) { mrow[i][rr] = rowmap[(slot0 + i) * 8 + r]; });
    acc.foreach_tile(wc, lane, [&](int i, int rr, int e, T(&tile)[PV][EW]) {
      const int m = mrow[i][rr];
      if (m < 0) return;
#pragma unroll
      for (int v = 0; v < PV; ++v) {
        T *val = tile[v];
        T *cp = Cb + (long long)m * ldc + v * cm.vstride + e;
        const long long room = interior ? EW : cm.lim - (vb + v * cm.vlim + e);
        if (room >= EW) {
          T out[EW];
          if (c2 != T(0)) {
#pragma unroll
            for (int j = 0; j < EW; ++j) out[j] = fma(c1, val[j], c2 * cp[j]);
          } else {
#pragma unroll
            for (int j = 0; j < EW; ++j) out[j] = c1 * val[j];
          }
          if (EW == 2 && sizeof(T) == 8) *reinterpret_cast<double2 *>(cp) = *reinterpret_cast<double2 *>(out);
          else if (EW == 2) *reinterpret_cast<float2 *>(cp) = *reinterpret_cast<float2 *>(out);
          else cp[0] = out[0];
        } else {
#pragma unroll
          for (int j = 0; j < EW; ++j)
            if (j < room) cp[j] = (c2 != T(0)) ? fma(c1, val[j], c2 * cp[j]) : c1 * val[j];
        }
      }
    });
  }
};

// ---- the persistent main loop.  Grid = any number of CTAs; CTA b owns panels b, b+grid, ...
template <typename T, int NIT, int CX, class Prod, class Epi>
__device__ __forceinline__ void panel_mainloop(const PanelOp<T> &op, const Prod &prod_in, const Epi &epi, long long npanels_per_batch,
                                               int nbatch, char *smem) {
  // A CTA holds NG (1 or 2) independent warp groups.  Each group owns its own accumulators, its own cp.async ring and its own
  // stream of panels; they share only the operator image.  Group 1 starts half a panel late, so that one group's epilogue
  // (global loads and stores, latency-bound) and chunk waits run under the other group's multiplies.
  const int WC = op.WC, NS = op.NS, NE = op.NE, NG = op.NG;
  const int nthreads = 32 * op.WR * WC;              // threads of one group
  const int grp = threadIdx.x / nthreads;
  const int tid = threadIdx.x - grp * nthreads, lane = tid & 31, warp = tid >> 5;
  Prod prod(prod_in);
  prod.init(NE, tid, nthreads);
  const int wr = warp / WC, wc = warp - wr * WC;
  const int LDB = PV * NE + 4;
  OpSmem<T> A;
  char *ringp = op_smem_carve(smem, op, A);
  op_smem_load(smem, op, threadIdx.x, blockDim.x);
  pcp_commit();
  const size_t stage_elems = (size_t)op.stage_elems;
  T *ring = reinterpret_cast<T *>(ringp) + (size_t)grp * PANEL_NSTAGE * stage_elems;
  const long long ntot = npanels_per_batch * nbatch;
  const long long first = (long long)blockIdx.x * NG + grp, stride = (long long)gridDim.x * NG;
  const long long mine = first < ntot ? (ntot - first + stride - 1) / stride : 0;
  const int nchunks = op.nchunks;
  const long long total = mine * nchunks;
  auto group_barrier = [&]() {
    if (NG == 1) __syncthreads();
    else asm volatile("bar.sync %0, %1;" ::"r"(1 + grp), "r"(nthreads) : "memory");
  };
  // two cursors over (panel, chunk): one for the loads being issued, one for the chunk being multiplied
  long long ipl = first, cpl = first;
  int ic = 0, cc = 0, istage = 0, cstage = 0;
  long long ibatch = ipl / npanels_per_batch;
  ipl -= ibatch * npanels_per_batch;
  long long cbatch = ibatch;
  cpl = ipl;
  bool image_ready = false;                          // the shared operator image (with the chunk table) has landed
  auto issue = [&]() {
    // chunk table: from shared memory once it is there -- a global read here sits on the critical path of every chunk
    const ChunkDesc cd = image_ready ? A.chunks[ic] : op.chunks[ic];
    prod.issue(cd, ibatch, ipl, ring + istage * stage_elems, LDB, NE, tid, nthreads);
    if (++istage == PANEL_NSTAGE) istage = 0;
    if (++ic == nchunks) {
      ic = 0;
      ipl += stride;
      while (ipl >= npanels_per_batch) {
        ipl -= npanels_per_batch;
        ++ibatch;
      }
    }
  };
  for (int q = 0; q < PANEL_NSTAGE - 1; ++q) {
    if (q < total) issue();
    pcp_commit();
  }
  // the operator image was copied by all threads of the CTA: everyone's share must have landed before anyone reads it
  pcp_wait<PANEL_NSTAGE - 1>();
  __syncthreads();
  image_ready = true;
  const long long stagger_q = total > 0 ? (nchunks / 2 < total ? nchunks / 2 : total - 1) : -1;
  if (NG == 2) {
    if (grp == 1) asm volatile("bar.sync 3, %0;" ::"r"(2 * nthreads) : "memory");
    else if (stagger_q < 0) asm volatile("bar.arrive 3, %0;" ::"r"(2 * nthreads) : "memory");
  }
  Acc<T, NIT, CX> acc;
  acc.zero();
  for (long long q = 0; q < total; ++q) {
    pcp_wait<PANEL_NSTAGE - 2>();
    group_barrier();
    if (q + PANEL_NSTAGE - 1 < total) issue();
    pcp_commit();
    T *stage = ring + cstage * stage_elems;
    if (Prod::kTransform) {
      const ChunkDesc cd = A.chunks[cc];
      if (cd.kind != KIND_PLAIN) {                   // uniform over the group
        prod.transform(cd, cbatch, cpl, stage, LDB, NE, tid, nthreads);
        group_barrier();
      }
    }
    // the epilogue's own global operands: pull them into L2 while the last chunk is multiplied
    if (cc == nchunks - 1 && !(op.dbg & 4)) epi.prefetch(acc, A.rowmap, wr * NIT, cbatch, cpl, wc, lane);
    if (!(op.dbg & 1)) {
      if (op.sparse) acc.mac_chunk(A, cc, NS, wr * NIT, stage, LDB, NE, wc, lane);
      else acc.mac_dense(A, A.chunks[cc], NS, wr * NIT, stage, LDB, NE, wc, lane);
    }
    if (NG == 2 && grp == 0 && q == stagger_q) asm volatile("bar.arrive 3, %0;" ::"r"(2 * nthreads) : "memory");
    if (++cstage == PANEL_NSTAGE) cstage = 0;
    if (++cc == nchunks) {
      if (!(op.dbg & 2)) epi(acc, A.rowmap, wr * NIT, cbatch, cpl, wc, lane);
      acc.zero();
      cc = 0;
      cpl += stride;
      while (cpl >= npanels_per_batch) {
        cpl -= npanels_per_batch;
        ++cbatch;
      }
    }
  }
  pcp_wait<0>();
}

// Dispatch over the compile-time accumulator shapes.  FP64: NIT*CX <= 8; FP32: NIT*CX <= 4.
#define FR_PANEL_SHAPES_F64(X) \
  X(1, 1) X(2, 1) X(3, 1) X(4, 1) X(5, 1) X(6, 1) X(7, 1) X(8, 1) X(1, 2) X(2, 2) X(3, 2) X(4, 2)
#define FR_PANEL_SHAPES_F32(X) X(1, 1) X(2, 1) X(3, 1) X(4, 1) X(1, 2) X(2, 2)
// triple-packed operators (gradient): NIT a multiple of 3
#define FR_PANEL_TRIPLES_F64(X) X(3, 1) X(6, 1) X(3, 2)
#define FR_PANEL_TRIPLES_F32(X) X(3, 1)

template <typename T>
inline size_t panel_smem_bytes(const PanelOp<T> &op) {
  return op.smem_op + (size_t)op.NG * PANEL_NSTAGE * op.stage_elems * sizeof(T) + 16;
}

}  // namespace frb
