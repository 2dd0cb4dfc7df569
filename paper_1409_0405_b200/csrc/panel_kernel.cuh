// The persistent, warp-specialised panel main loop shared by the plain operator product and its fused variants (panel.cuh).
//
// Warps of a CTA:  [group 0 consumers | group 1 consumers | ... | one producer warp per group].
//   producer (one elected lane): for every (panel, chunk) of its group, wait until the ring stage is empty, arm the stage's
//     full barrier with the byte count and issue the tiled copy/copies (cp.async.bulk.tensor) that fill it;
//   consumers: wait on the full barrier, multiply the chunk into their register accumulators, release the stage (one arrive
//     per warp on the empty barrier), and after the panel's last chunk run the epilogue on their own rows and columns.
// No warp ever waits for another consumer warp: a warp in its (latency-bound) epilogue leaves the tensor pipe to the warps that
// are already multiplying the next panel, as far ahead as the ring is deep.  In plans with one warp group whose consumer warps are
// not a multiple of four, the warps do not even keep a fixed (row, column) role: they take (panel, role) units from a counter (DYN).
#pragma once
#include "panel.cuh"
#include "tma.cuh"

namespace frb {

// Where a panel's columns live in a global matrix: column(v, e) = p*pstride + v*vstride + e, valid iff
// p*pstride + v*vlim + e < lim.  State matrices [rows][5][ld]: pstride = NE, vstride = ld, vlim = 0, lim = ld.
// Plain matrices [rows][N] (fr_gemm): pstride = 5*NE, vstride = vlim = NE, lim = N.
struct ColMap {
  long long pstride, vstride, vlim, lim;
};

// ---- producer: B chunks are rows of up to two stacked global matrices, described by tensor maps (tma.cuh)
template <typename T>
struct alignas(64) TmaProducer {
  CUtensorMap tm[PANEL_MAXSRC];
  int plain;   // 1: plain matrix [K][N] (one copy per column block); 0: state matrix [rows][5][ld] (one copy per chunk)
  int pad[15];
  // called by one lane; `this` must be the kernel's __grid_constant__ parameter (the TMA unit reads the map through its address)
  __device__ __forceinline__ void issue(const ChunkDesc &cd, long long batch, long long pl, uint32_t dst, uint32_t bar, int NE) const {
    const CUtensorMap *m = &tm[cd.src];
    if (!plain) {
      if (sizeof(T) == 8) tma_load_4d(dst, m, 0, cd.row0, (int)(pl * (NE >> 4)), 0, bar);
      else tma_load_3d(dst, m, (int)(pl * NE), cd.row0, 0, bar);
    } else if (sizeof(T) == 8) {
      const int nb = PV * (NE >> 4);
      const uint32_t pp = (uint32_t)cd.step * 128u;
      const int col0 = (int)(pl * PV * NE);
      for (int j = 0; j < nb; ++j) tma_load_3d(dst + j * pp, m, col0 + j * 16, cd.row0, (int)batch, bar);
    } else {
      const uint32_t pp = (uint32_t)cd.step * (uint32_t)NE * 4u;
      const int col0 = (int)(pl * PV * NE);
#pragma unroll
      for (int v = 0; v < PV; ++v) tma_load_3d(dst + v * pp, m, col0 + v * NE, cd.row0, (int)batch, bar);
    }
  }
};

// ---- epilogue: C <- c1*acc + c2*C.  `plain` (decided on the host: c1 == 1 and c2 == 0, the case of every product inside fr_rhs)
// stores the accumulators as they are: no FP64 instruction in the epilogue, which would queue behind the other warps' DMMAs.
template <typename T>
struct PlainEpilogue {
  static constexpr bool kProducerPrefetch = false;
  T *C;
  long long ldc, bstride;
  ColMap cm;
  T c1, c2;
  int plain;
  template <typename ACC>
  __device__ __forceinline__ void prefetch(ACC &acc, const int *rowmap, int slot0, long long batch, long long pl, int wc,
                                           int lane) const {
    if (plain || c2 == T(0)) return;
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
    if (plain && interior) {
      acc.foreach_tile(wc, lane, [&](int i, int rr, int e, T(&tile)[PV][EW]) {
        const int m = mrow[i][rr];
        if (m < 0) return;
        T *cp = Cb + (long long)m * ldc + e;
#pragma unroll
        for (int v = 0; v < PV; ++v) {
          if (EW == 2 && sizeof(T) == 8) *reinterpret_cast<double2 *>(cp) = *reinterpret_cast<double2 *>(tile[v]);
          else if (EW == 2) *reinterpret_cast<float2 *>(cp) = *reinterpret_cast<float2 *>(tile[v]);
          else cp[0] = tile[v][0];
          cp += cm.vstride;
        }
      });
      return;
    }
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

// ---- the persistent main loop.  Grid = any number of CTAs; CTA b, group g owns panels b*NG+g, b*NG+g + grid*NG, ...
// `prod` must refer to the kernel's __grid_constant__ parameter.
// STREAM: the operator's packed blocks travel through the ring (PanelOp::stream; plain products only -- a compile-time switch so that
// the kernels of resident operators carry none of it).
// DYN (one warp group): the consumer warps take (panel, warp role) units from a shared counter instead of keeping a fixed role.  The
// FP64 tensor pipe is per SM sub-partition, and ten consumer warps sit 3/3/2/2 on the four of them: with fixed roles the warps of the
// crowded sub-partitions set the pace and the others wait at the ring; with units, a warp that runs faster simply takes more of them.
// Results do not depend on which warp computes a unit.
template <typename T, int NIT, int CX, class Prod, class Epi, bool PACKED = true, bool STREAM = false, bool DYN = false>
__device__ __forceinline__ void panel_mainloop(const PanelOp<T> &op, const Prod &prod, const Epi &epi, long long npanels_per_batch,
                                               int nbatch, char *smem_raw) {
  const int WC = op.WC, NS = op.NS, NE = op.NE, NG = op.NG;
  const int nwc = op.WR * WC;                          // consumer warps of one group
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const bool producer = warp >= nwc * NG;
  const int grp = producer ? warp - nwc * NG : warp / nwc;
  const int nstage = op.nstage;
  // ---- carve shared memory: operator image | ring (1024-byte aligned: the swizzle is a function of the address) | barriers
  const uint32_t s0 = smem_u32(smem_raw);
  const uint32_t ring0 = (s0 + (uint32_t)op.smem_op + 1023u) & ~1023u;
  char *ringp = smem_raw + (ring0 - s0);
  const uint32_t stage_bytes = (uint32_t)op.stage_bytes;
  const uint32_t bars = ring0 + (uint32_t)(NG * nstage) * stage_bytes;
  // barriers: full[g][s] at bars + (g*nstage + s)*16, empty[g][s] 8 bytes later; the image barrier closes the list
  const uint32_t bar_img = bars + (uint32_t)(NG * nstage) * 16u;
  if (threadIdx.x == 0) {
    for (int i = 0; i < NG * nstage; ++i) {
      mbar_init(bars + i * 16, 1);
      mbar_init(bars + i * 16 + 8, (uint32_t)nwc);
    }
    mbar_init(bar_img, 1);
    mbar_fence_init();
    if (DYN) *reinterpret_cast<int *>(smem_raw + (bar_img + 16u - s0)) = 0;   // the unit counter
  }
  __syncthreads();
  OpSmem<T> A;
  op_smem_carve(smem_raw, op, A);
  // panel counts fit 32 bits (leading dimensions are below 2^31 and a panel has at least 16 elements)
  const int npb = (int)npanels_per_batch;
  const long long ntot = npanels_per_batch * nbatch;
  const int first = blockIdx.x * NG + grp, stride = gridDim.x * NG;
  const int mine = first < ntot ? (int)((ntot - first + stride - 1) / stride) : 0;
  const int nchunks = op.nchunks;
  const int total = mine * nchunks;
  const uint32_t gbar = bars + (uint32_t)(grp * nstage) * 16u;
  const uint32_t gring = ring0 + (uint32_t)(grp * nstage) * stage_bytes;

  if (producer) {
    if (lane != 0) return;
    if (grp == 0) {
      // the operator image: five bulk copies counted on one barrier
      mbar_expect_tx(bar_img, (uint32_t)op.smem_op);
      uint32_t d = s0;
      if (!STREAM) bulk_load(d, op.vals, (uint32_t)op.bytes_vals, bar_img);   // a streamed operator keeps no blocks here
      d += (uint32_t)op.bytes_vals;
      bulk_load(d, op.idx, (uint32_t)op.bytes_idx, bar_img);
      d += (uint32_t)op.bytes_idx;
      bulk_load(d, op.off, (uint32_t)op.bytes_off, bar_img);
      d += (uint32_t)op.bytes_off;
      bulk_load(d, op.rowmap, (uint32_t)op.bytes_rowmap, bar_img);
      d += (uint32_t)op.bytes_rowmap;
      bulk_load(d, op.chunks, (uint32_t)op.bytes_chunks, bar_img);
    }
    int pl = first, batch = pl / npb;
    pl -= batch * npb;
    int stage = 0;
    uint32_t phase = 0;
    const uint32_t ablk = (uint32_t)NS * (sizeof(T) == 8 ? 256u : 32u);   // bytes of one packed block row (all slots)
    for (int p = 0; p < mine; ++p) {
      for (int c = 0; c < nchunks; ++c) {
        const ChunkDesc cd = op.chunks[c];               // global (L1-resident); the image may not have landed yet
        mbar_wait(gbar + stage * 16 + 8, phase ^ 1u);    // stage is empty
        const uint32_t full = gbar + stage * 16;
        // streamed operator: the chunk's packed blocks follow its rows of B into the stage (one bulk copy, L2-resident source)
        const uint32_t abytes = STREAM ? (uint32_t)cd.nblk * ablk : 0u;
        mbar_expect_tx(full, (uint32_t)(PV * NE * (int)sizeof(T)) * (uint32_t)cd.step + abytes);
        prod.issue(cd, batch, pl, gring + stage * stage_bytes, full, NE);
        if (STREAM)
          bulk_load(gring + stage * stage_bytes + (uint32_t)op.a_off(), reinterpret_cast<const char *>(op.vals) + (size_t)cd.base * ablk, abytes, full);
        // with the panel's last chunk on its way, pull what its epilogue will read into L2 (epilogues that have tensor maps for it)
        if constexpr (Epi::kProducerPrefetch) {
          if (c == nchunks - 1) epi.producer_prefetch(pl);
        }
        if (++stage == nstage) {
          stage = 0;
          phase ^= 1u;
        }
      }
      pl += stride;
      while (pl >= npb) {
        pl -= npb;
        ++batch;
      }
    }
    return;
  }

  // ---- consumers
  const int tid = threadIdx.x - grp * nwc * 32;
  const int cw = tid >> 5;                             // warp within the group
  const int wr = cw / WC, wc = cw - wr * WC;
  mbar_wait(bar_img, 0);
  int cpl = first, cbatch = cpl / npb;
  cpl -= cbatch * npb;
  // Group 1 starts half a panel late, so that one group's epilogue (global loads and stores, latency-bound) runs under the
  // other group's multiplies.
  const int stagger_q = total > 0 ? (nchunks / 2 < total ? nchunks / 2 : total - 1) : -1;
  if (NG == 2) {
    if (grp == 1) asm volatile("bar.sync 3, %0;" ::"r"(2 * nwc * 32) : "memory");
    else if (stagger_q < 0) asm volatile("bar.arrive 3, %0;" ::"r"(2 * nwc * 32) : "memory");
  }
  Acc<T, NIT, CX, PACKED> acc;
  acc.zero();
  if constexpr (DYN) {
    int *ctr = reinterpret_cast<int *>(smem_raw + (bar_img + 16u - s0));
    const int nunits = mine * nwc;
    for (;;) {
      int U = 0;
      if (lane == 0) U = atomicAdd(ctr, 1);
      U = __shfl_sync(0xffffffffu, U, 0);
      if (U >= nunits) break;
      const int pi = U / nwc, role = U - pi * nwc;         // panel of this CTA's sequence, warp role in it
      const int uwr = role / WC, uwc = role - uwr * WC;
      const long long pabs = (long long)first + (long long)pi * stride;
      const int ubatch = (int)(pabs / npb), upl = (int)(pabs - (long long)ubatch * npb);
      for (int c = 0; c < nchunks; ++c) {
        const int q = pi * nchunks + c;                    // the chunk's number in the ring: stage and phase follow from it
        const int stg = q % nstage;
        mbar_wait(gbar + stg * 16, (uint32_t)(q / nstage) & 1u);
        const char *st = ringp + (size_t)stg * stage_bytes;
        if (c == 0 && op.pf_epi) epi.prefetch(acc, A.rowmap, uwr * NIT, ubatch, upl, uwc, lane);
        if (op.sparse) acc.mac_chunk(A, c, A.chunks[c], NS, uwr * NIT, st, NE, uwc, lane);
        else acc.template mac_dense<STREAM>(A, A.chunks[c], NS, uwr * NIT, st, NE, uwc, lane, STREAM ? op.a_off() : 0);
        __syncwarp();
        if (lane == 0) mbar_arrive(gbar + stg * 16 + 8);
      }
      epi(acc, A.rowmap, uwr * NIT, ubatch, upl, uwc, lane);
      acc.zero();
    }
    return;
  }
  int stage = 0, cc = 0;
  uint32_t phase = 0;
  for (int q = 0; q < total; ++q) {
    mbar_wait(gbar + stage * 16, phase);
    const char *st = ringp + (size_t)(grp * nstage + stage) * stage_bytes;
    // the epilogue's own global operands: pull them into L2 while the panel is multiplied
    if (cc == 0 && op.pf_epi) epi.prefetch(acc, A.rowmap, wr * NIT, cbatch, cpl, wc, lane);
#ifdef FRB_DEBUG_KNOBS
    if (!(op.dbg & 1))
#endif
    {
      if (op.sparse) acc.mac_chunk(A, cc, A.chunks[cc], NS, wr * NIT, st, NE, wc, lane);
      else acc.template mac_dense<STREAM>(A, A.chunks[cc], NS, wr * NIT, st, NE, wc, lane, STREAM ? op.a_off() : 0);
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(gbar + stage * 16 + 8);
    if (NG == 2 && grp == 0 && q == stagger_q) asm volatile("bar.arrive 3, %0;" ::"r"(2 * nwc * 32) : "memory");
    if (++stage == nstage) {
      stage = 0;
      phase ^= 1u;
    }
    if (++cc == nchunks) {
#ifdef FRB_DEBUG_KNOBS
      if (!(op.dbg & 2))
#endif
      epi(acc, A.rowmap, wr * NIT, cbatch, cpl, wc, lane);
      acc.zero();
      cc = 0;
      cpl += stride;
      while (cpl >= npb) {
        cpl -= npb;
        ++cbatch;
      }
    }
  }
}

// Units (DYN) pay an atomic and an index computation per unit: worth it where fixed roles leave the sub-partitions unevenly loaded,
// i.e. where the consumer warps of the one group are not a multiple of four.  FRB_NO_DYN=1: fixed roles everywhere.
template <typename T>
inline bool panel_use_units(const PanelOp<T> &op) {
  return op.NG == 1 && (op.WR * op.WC) % 4 != 0 && getenv("FRB_NO_DYN") == nullptr;
}

// Dispatch over the compile-time accumulator shapes.  FP64: NIT*CX <= 8; FP32: NIT*CX <= 4.
#define FR_PANEL_SHAPES_F64(X) \
  X(1, 1) X(2, 1) X(3, 1) X(4, 1) X(5, 1) X(6, 1) X(7, 1) X(8, 1) X(1, 2) X(2, 2) X(3, 2) X(4, 2)
#define FR_PANEL_SHAPES_F32(X) X(1, 1) X(2, 1) X(3, 1) X(4, 1) X(1, 2) X(2, 2)
// triple-packed operators (gradient): NIT a multiple of 3
#define FR_PANEL_TRIPLES_F64(X) X(3, 1) X(6, 1) X(3, 2)
#define FR_PANEL_TRIPLES_F32(X) X(3, 1)

// grid: one CTA per SM and CTA slot, never more than there are panel sets.  The opt-in to > 48 kB of dynamic shared memory is a
// per-device function attribute; setting it on every launch keeps the launchers free of process-wide state (it is not a stream
// operation, so it is legal under capture).
template <typename T, typename K, typename A>
inline void panel_launch(K k, const A &a, const PanelOp<T> &op, long long ntot, cudaStream_t s) {
  const size_t smem = panel_smem_bytes(op);
  FR_CUDA_TRY(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  const int nthreads = 32 * (op.WR * op.WC * op.NG + op.NG);
  const long long grid = std::min<long long>((ntot + op.NG - 1) / op.NG, (long long)device_sm_count() * op.occ);
  k<<<(unsigned)grid, nthreads, smem, s>>>(a);
  FR_CUDA_TRY(cudaGetLastError());
}

}  // namespace frb
