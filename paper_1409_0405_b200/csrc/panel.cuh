// Panel kernels: the operator products C <- c1*A*B + c2*C (eq. 1) and their fusions with the adjacent
// point-wise work, for one element type.  "A is a constant operator matrix, and B and C are row-major state matrices"
// (PAPER.md:39): every column of B is independent, so one CTA owns a *panel* of NE consecutive elements (all 5
// conserved variables = 5*NE columns) and ALL rows of A -- the column slicing the paper's OpenMP backend found best
// -- while B streams through shared memory in K-chunks and the accumulators stay in registers.
//
// B200 design:
//   * the operator is packed once at fr_setup into 8-row groups with a compact list of the k indices that are non-zero
//     in the group (dense operators: all k; prism operators are 15-45 % dense and skip the rest) and stays resident in
//     shared memory for the life of the persistent CTA;
//   * FP64 multiplies on the FP64 tensor pipe, mma.sync.m8n8k4.f64 (DMMA: measured 37.1 TFLOP/s on B200 against 33.7
//     for a DFMA chain, with 1/8 of the issue slots and a fraction of the shared-memory operand traffic);
//     FP32 multiplies with FFMA on register tiles of 8 rows x 5 variables x (1|2) elements (no TF32: the 2e-5 parity
//     bound excludes it, and tcgen05 has no FP32/FP64 kind);
//   * B chunks arrive through a multi-stage cp.async ring that runs across panel boundaries; rows are padded so that the
//     DMMA fragment loads are bank-conflict free;
//   * producers (how a B chunk comes to be) and epilogues (what happens to the accumulators) are policies, which is how the
//     point-wise flux, gradient transform, -1/|J| scaling and Runge-Kutta stage update are fused into the products.
#pragma once
#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <numeric>

#include "common.cuh"

namespace frb {

constexpr int PV = FR_NVAR;          // variable segments per panel
constexpr int PANEL_MAXW = 16;       // warps per CTA (upper bound; 8 when the accumulators need > 128 registers)
constexpr int PANEL_MAXCHUNKS = 64;
#ifndef FRB_NSTAGE
#define FRB_NSTAGE 2
#endif
constexpr int PANEL_NSTAGE = FRB_NSTAGE;   // cp.async ring depth: 2 beats 3 and 4 on config 3 (taller chunks, fewer barriers; profiles/r01_c_fusion_notes.md)

// One K-chunk of the stacked right-hand operand: rows [row0, row0+nrows) of source `src`.
struct ChunkDesc {
  int src, row0, nrows, kind;
  int base, pad0, pad1, pad2;   // dense operators: first packed block (FP64: 4 rows) / row (FP32) of this chunk
};

// Device image of a packed operator + its launch geometry (all pointers device).
template <typename T>
struct PanelOp {
  int M = 0, K = 0;
  int WR = 0, WC = 0, NIT = 0, CX = 0;   // warp grid, row groups per row-warp, column blocks (FP64) / elements per lane (FP32)
  int NE = 0;                            // elements per panel (of one warp group)
  int NG = 1;                            // independent warp groups per CTA, each streaming its own panels (staggered)
  int occ = 1;                           // CTAs per SM the plan was sized for (shared memory and registers)
  int KC = 0, nchunks = 0, NS = 0;       // rows per chunk (max), chunks, slots = WR*NIT
  int stage_elems = 0;                   // elements of one ring stage
  int curved = 0;                        // flux chunks: metric terms per point (1) or per element (0)
  int nblk = 0;                          // packed blocks (FP64: 8x4 tiles; FP32: 8x1 columns)
  int nidx = 0;                          // entries of idx
  int dbg = 0;                           // measurement aid (env FRB_PANEL_DBG): 1 skip multiply, 2 skip epilogue
  int sparse = 0;                        // 1: per-group k-lists (idx/off); 0: dense, all slots share the chunk's rows
  double macs_per_col = 0;               // executed multiply-adds per column (dense: M*K)
  double density = 1;                    // fraction of non-zero entries of the operator
  T *vals = nullptr;                     // FP64 [nblk][32]; FP32 [nblk][8]
  uint32_t *idx = nullptr;               // byte offset of the B row in the stage: FP64 [nblk][4], FP32 [nblk]
  int *off = nullptr;                    // [nchunks*NS + 1]
  int *rowmap = nullptr;                 // [NS*8] actual row of (slot, r) or -1
  ChunkDesc *chunks = nullptr;           // [nchunks]
  size_t smem_op = 0;                    // bytes of the operator image in shared memory
  bool ok() const { return vals != nullptr; }
};

template <typename T>
void panel_op_free(PanelOp<T> &p) {
  if (p.vals) cudaFree(p.vals);
  if (p.idx) cudaFree(p.idx);
  if (p.off) cudaFree(p.off);
  if (p.rowmap) cudaFree(p.rowmap);
  if (p.chunks) cudaFree(p.chunks);
  p = PanelOp<T>();
}

// How the K dimension of the operator is fed: a list of sources stacked along K, each cut into chunks of at most KC rows.
// kind 0: `rows` plain rows of a global matrix <-> `rows` columns of A.
// kind 1 (kept for producers that transform a chunk in shared memory -- kTransform in panel_kernel.cuh; not used by the kernels of
//         this round, see panel_fused.cu for why): transformed flux at `rows` solution points <-> 3*rows columns of A (alpha-major: column alpha*rows + nu); a chunk
//         of n points occupies stage rows [0,3n) (alpha-major within the chunk: row alpha*n + j) for G -> F~, rows [3n,4n)
//         for U, followed by the metric terms (flux_stage_elems).
struct KSource {
  int rows;
  int kind;
  int unit;      // unused (kept for aggregate initialisation)
};
constexpr int KIND_PLAIN = 0, KIND_FLUX = 1;

// shared-memory elements of one stage holding a flux chunk of n points
inline __host__ __device__ size_t flux_stage_elems(int n, int NE, int LDB, int curved) {
  return (size_t)4 * n * LDB + (size_t)9 * (curved ? n : 1) * NE;
}

struct PanelGeom {
  int WR, WC, NIT, CX, NE;
  double eff;
  int NG;
  int occ;
};

// Warps per CTA a given accumulator shape allows: registers per thread ~ accumulators + 70 must fit the 64K register file.
// FP64: NIT*CX*10 doubles per thread; FP32: NIT*CX*40 floats.
template <typename T>
constexpr int panel_maxw(int nit, int cx) {
  // FP32 tiles also keep 8 operator values and 5*CX state values live per k and index more arrays: with only +70 registers of
  // head-room the CX = 2 shapes spilled inside the multiply loop (8x slower), so FP32 with CX = 2 budgets +110.
  const int acc_regs = sizeof(T) == 8 ? nit * cx * 20 : nit * cx * 40;
  const int w = 2048 / (acc_regs + ((sizeof(T) == 4 && cx == 2) ? 110 : 70));
  return w > 16 ? 16 : (w < 1 ? 1 : w);
}

// Choose the warp grid for G row groups.  The FP64 tensor pipe takes one DMMA per warp every ~32 cycles, so two warps per
// scheduler saturate it only if they do nothing else: prefer 12-16 warps per SM.
template <typename T>
inline std::vector<PanelGeom> list_geoms(int G, int min_ne, int max_ne, int triple, bool dense) {
  std::vector<PanelGeom> all;
  const bool f64 = sizeof(T) == 8;
  const int gu = triple ? 3 : 1;            // groups come in units of `gu` that must stay on one row-warp
  const int GU = (G + gu - 1) / gu;
  // two groups help some FP64 kernels and hurt most FP32 ones (profiles/r01_c_fusion_notes.md): both are candidates, the static
  // score favours them in FP64 only, and the autotuner decides on large meshes
  const int ngmax = getenv("FRB_PANEL_NG") ? atoi(getenv("FRB_PANEL_NG")) : 2;
  // FRB_MIN_EFF: row-warps without rows still issue copies, which can pay (profiles/r01_j_panel_source_level.md)
  const double min_eff = getenv("FRB_MIN_EFF") ? atof(getenv("FRB_MIN_EFF")) : 0.7;
  for (int NG = 1; NG <= ngmax; ++NG)
    for (int WR = 1; WR <= PANEL_MAXW; ++WR) {
      const int nit = ((GU + WR - 1) / WR) * gu;
      for (int WC = 1; NG * WR * WC <= PANEL_MAXW; WC *= 2) {
        for (int CX = 2; CX >= 1; --CX) {
          if (f64 ? nit * CX > 8 : nit * CX > 4) continue;
          const int W = NG * WR * WC;
          if (W > panel_maxw<T>(nit, CX)) continue;
          const int NE = (f64 ? 8 : 32) * CX * WC;
          if (NE < min_ne || NE > max_ne) continue;
          double eff = (double)G / (WR * nit);
          if (eff < min_eff) continue;                   // more than 30 % of the row slots empty: not timed by default
          // prefer many warps, then wider panels, then fewer accumulators
          double score = eff * (0.4 + 0.6 * std::min(W, 14) / 14.0) * (1.0 + 0.02 * std::log2((double)NE)) * (1.0 - 0.005 * nit * CX);
          // dense operators: the B fragments of a k-block are shared by the NIT row groups of the warp; shared-memory
          // wavefronts per multiply ~ 2/NIT + 0.4/CX
          if (dense) score /= 1.0 + 0.4 * (2.0 / nit + 0.4 / CX);
          // two staggered warp groups hide one group's epilogue and load waits behind the other's multiplies
          if (NG == 2) score *= f64 ? 1.25 : 0.85;
          all.push_back(PanelGeom{WR, WC, nit, CX, NE, score, NG, 1});
          // two CTAs per SM (half the shared memory and registers each): another way to overlap one panel's epilogue and
          // load waits with another's multiplies; only timing (fr_setup autotuning) tells which wins
          if (NG == 1 && 2 * W <= panel_maxw<T>(nit, CX)) all.push_back(PanelGeom{WR, WC, nit, CX, NE, score * 0.9, NG, 2});
        }
      }
    }
  std::stable_sort(all.begin(), all.end(), [](const PanelGeom &x, const PanelGeom &y) { return x.eff > y.eff; });
  return all;
}

// Best geometry by the static score; fr_setup may instead time the first few candidates on the real arrays (PackOptions::cand).
template <typename T>
inline PanelGeom choose_geom(int G, int min_ne, int max_ne, int triple, bool dense, int cand = 0) {
  const std::vector<PanelGeom> all = list_geoms<T>(G, min_ne, max_ne, triple, dense);
  if (cand < 0 || cand >= (int)all.size()) return PanelGeom{0, 0, 0, 0, 0, -1.0, 1, 1};
  return all[cand];
}

// Greedy clustering of rows into groups of 8 with similar column support (sparse operators only).
inline std::vector<int> cluster_rows(const std::vector<std::vector<uint8_t>> &sup, int M, int K) {
  std::vector<int> order;
  std::vector<char> used(M, 0);
  std::vector<int> cnt(M, 0);
  for (int m = 0; m < M; ++m)
    for (int k = 0; k < K; ++k) cnt[m] += sup[m][k];
  int remaining = M;
  while (remaining > 0) {
    // seed: the unused row with the largest support
    int seed = -1;
    for (int m = 0; m < M; ++m)
      if (!used[m] && (seed < 0 || cnt[m] > cnt[seed])) seed = m;
    std::vector<uint8_t> u = sup[seed];
    used[seed] = 1;
    order.push_back(seed);
    --remaining;
    for (int j = 1; j < 8 && remaining > 0; ++j) {
      int bi = -1;
      int bgrow = 1 << 30, bshare = -1;
      for (int m = 0; m < M; ++m) {
        if (used[m]) continue;
        int grow = 0, share = 0;
        for (int k = 0; k < K; ++k) {
          grow += sup[m][k] & ~u[k] & 1;
          share += sup[m][k] & u[k];
        }
        if (grow < bgrow || (grow == bgrow && share > bshare)) {
          bgrow = grow;
          bshare = share;
          bi = m;
        }
      }
      used[bi] = 1;
      order.push_back(bi);
      --remaining;
      for (int k = 0; k < K; ++k) u[k] |= sup[bi][k];
    }
    while (order.size() % 8) order.push_back(-1);
  }
  return order;
}

struct PackOptions {
  int min_ne = 16, max_ne = 64;
  int triple = 0;          // rows come as (alpha, rho) with alpha-major blocks of M/3: keep the three alpha of a rho in one thread
  int kc = 0;              // rows per chunk (0 = default)
  int allow_sparse = 1;
  int curved = 0;          // flux sources: per-point metric terms
  int cand = 0;            // k-th best geometry by static score (autotuning)
  const int *row_ids = nullptr;   // row split: the epilogue's row number of each row of A (nullptr = 0..M-1)
};

// Pack A (M x K, host FP64, row-major) for the panel kernels.  `srcs` stacks the K dimension.  Returns false if the
// operator does not fit the resident-in-shared-memory design (caller falls back to the streaming kernel).
template <typename T>
bool panel_op_build_kc(PanelOp<T> &p, int M, int K, const double *A, const std::vector<KSource> &srcs, const PackOptions &opt,
                       size_t smem_budget, size_t smem_total, int kc_try, int *kc_fit);

// Chunk height: as tall as the B ring allows (few, large cp.async stages keep enough bytes in flight to cover HBM latency
// with one persistent CTA per SM); first try whole sources, then the height that makes three stages fit `smem_total`.
template <typename T>
bool panel_op_build(PanelOp<T> &p, int M, int K, const double *A, const std::vector<KSource> &srcs, const PackOptions &opt,
                    size_t smem_budget, size_t smem_total = 220 * 1024) {
  // FRB_FORCE_CAND=k: build candidate k (geometry + 1000 * opposite packing) where the caller asked for the default; falls back
  // to the default if k does not exist for this operator.  Lets the parity tests cover every candidate the autotuner may pick.
  if (opt.cand == 0 && getenv("FRB_FORCE_CAND")) {
    PackOptions o2 = opt;
    o2.cand = atoi(getenv("FRB_FORCE_CAND"));
    if (o2.cand != 0 && panel_op_build(p, M, K, A, srcs, o2, smem_budget, smem_total)) return true;
  }
  int kc = opt.kc > 0 ? opt.kc : 252;
  for (int attempt = 0; attempt < 6 && kc >= 4; ++attempt) {
    int fit = 0;
    if (panel_op_build_kc(p, M, K, A, srcs, opt, smem_budget, smem_total, kc, &fit)) return true;
    if (fit <= 0) return false;
    kc = std::min(fit, kc - 4);
  }
  return false;
}

template <typename T>
bool panel_op_build_kc(PanelOp<T> &p, int M, int K, const double *A, const std::vector<KSource> &srcs, const PackOptions &opt,
                       size_t smem_budget, size_t smem_total, int kc_try, int *kc_fit) {
  const bool f64 = sizeof(T) == 8;
  int ktot = 0;
  for (auto &s : srcs) ktot += s.kind == KIND_FLUX ? 3 * s.rows : s.rows;
  FR_REQUIRE(ktot == K, "panel_op_build: sources do not add up to K");
  double amax = 0;
  for (size_t i = 0; i < (size_t)M * K; ++i) {
    FR_REQUIRE(A[i] == A[i] && A[i] - A[i] == 0.0, "operator contains non-finite entries");
    amax = std::max(amax, std::fabs(A[i]));
  }
  // structural zeros: entries below 2^-46 of the largest entry are dropped (reading R24)
  const double thr = amax * 1.4210854715202004e-14;
  std::vector<std::vector<uint8_t>> sup(M, std::vector<uint8_t>(K, 0));
  size_t nnz = 0;
  for (int m = 0; m < M; ++m)
    for (int k = 0; k < K; ++k)
      if (std::fabs(A[(size_t)m * K + k]) > thr) {
        sup[m][k] = 1;
        ++nnz;
      }
  const double density = (double)nnz / ((double)M * K);
  // automatic choice: k-lists below 60 % density; cand >= 1000 asks for the opposite packing (the autotuner times both for
  // operators of intermediate density, e.g. [M4 | M6] of tetrahedra, 66 % dense, whose M6 half is zero for two faces per alpha)
  const bool flip = opt.cand >= 1000 && density < 0.95;
  const bool sparse = (opt.allow_sparse && density < 0.6) != flip;
  // ---- rows -> groups of 8
  std::vector<int> order;   // virtual row -> actual row or -1
  if (opt.triple) {
    FR_REQUIRE(M % 3 == 0, "triple packing needs M divisible by 3");
    const int nu = M / 3;
    std::vector<int> rho_order;
    if (sparse) {
      std::vector<std::vector<uint8_t>> s3(nu, std::vector<uint8_t>(K, 0));
      for (int r = 0; r < nu; ++r)
        for (int a = 0; a < 3; ++a)
          for (int k = 0; k < K; ++k) s3[r][k] |= sup[a * nu + r][k];
      rho_order = cluster_rows(s3, nu, K);
    } else {
      for (int r = 0; r < nu; ++r) rho_order.push_back(r);
      while (rho_order.size() % 8) rho_order.push_back(-1);
    }
    // group 3g+a holds rows (a, rho_order[8g .. 8g+7])
    for (size_t g = 0; g < rho_order.size() / 8; ++g)
      for (int a = 0; a < 3; ++a)
        for (int r = 0; r < 8; ++r) {
          const int rho = rho_order[8 * g + r];
          order.push_back(rho < 0 ? -1 : a * nu + rho);
        }
  } else if (sparse) {
    order = cluster_rows(sup, M, K);
  } else {
    for (int m = 0; m < M; ++m) order.push_back(m);
    while (order.size() % 8) order.push_back(-1);
  }
  const int G = (int)order.size() / 8;
  // ---- chunks
  const int KC = kc_try;
  std::vector<ChunkDesc> chunks;
  std::vector<std::vector<int>> chunk_cols;   // column of A behind each MAC row of the chunk's stage
  {
    int k0 = 0, si = 0;
    for (auto &s : srcs) {
      if (s.kind == KIND_PLAIN) {
        // equal chunks of at most KC rows, a multiple of 4 so that dense k-lists need no padding
        const int nch = std::max(1, (s.rows + KC - 1) / KC);
        int step = ((s.rows + nch - 1) / nch + 3) / 4 * 4;
        if (step > KC) step = std::max(4, KC / 4 * 4);
        for (int r = 0; r < s.rows; r += step) {
          const int n = std::min(step, s.rows - r);
          chunks.push_back(ChunkDesc{si, r, n, s.kind, 0, 0, 0, 0});
          std::vector<int> cols(n);
          for (int j = 0; j < n; ++j) cols[j] = k0 + r + j;
          chunk_cols.push_back(cols);
        }
        k0 += s.rows;
      } else {
        const int nlim = std::max(1, KC / 3);
        const int nch = std::max(1, (s.rows + nlim - 1) / nlim);
        int step = (s.rows + nch - 1) / nch;
        if ((step + 3) / 4 * 4 <= nlim) step = (step + 3) / 4 * 4;
        for (int r = 0; r < s.rows; r += step) {
          const int n = std::min(step, s.rows - r);
          chunks.push_back(ChunkDesc{si, r, n, s.kind, 0, 0, 0, 0});
          std::vector<int> cols(3 * n);
          for (int a = 0; a < 3; ++a)
            for (int j = 0; j < n; ++j) cols[a * n + j] = k0 + a * s.rows + r + j;
          chunk_cols.push_back(cols);
        }
        k0 += 3 * s.rows;
      }
      ++si;
    }
  }
  const int nchunks = (int)chunks.size();
  if (nchunks > PANEL_MAXCHUNKS) return false;
  int kcmax = 0;
  for (auto &c : chunk_cols) kcmax = std::max(kcmax, (int)c.size());
  if (kcmax > 8000) return false;
  // ---- cost of each group (number of listed k) and its assignment to row-warps
  std::vector<std::vector<std::vector<int>>> lists(G, std::vector<std::vector<int>>(nchunks));
  std::vector<long long> gcost(G, 0);
  for (int g = 0; g < G; ++g)
    for (int c = 0; c < nchunks; ++c) {
      for (int kk = 0; kk < (int)chunk_cols[c].size(); ++kk) {
        bool any = !sparse;
        for (int r = 0; r < 8 && !any; ++r) {
          const int m = order[8 * g + r];
          if (m >= 0 && sup[m][chunk_cols[c][kk]]) any = true;
        }
        if (any) lists[g][c].push_back(kk);
      }
      const int n = (int)lists[g][c].size();
      gcost[g] += f64 ? (n + 3) / 4 * 4 : n;
    }
  PanelGeom geo = choose_geom<T>(G, opt.min_ne, opt.max_ne, opt.triple, !sparse, opt.cand % 1000);
  if (geo.eff < 0) return false;
  const int WR = geo.WR, NIT = geo.NIT, NS = WR * NIT;
  // LPT assignment of group units (1 or 3 groups) to row-warps, at most NIT groups per row-warp
  const int gu = opt.triple ? 3 : 1;
  const int GU = G / gu;
  std::vector<int> uorder(GU);
  std::iota(uorder.begin(), uorder.end(), 0);
  auto ucost = [&](int u) {
    long long c = 0;
    for (int j = 0; j < gu; ++j) c += gcost[u * gu + j];
    return c;
  };
  std::stable_sort(uorder.begin(), uorder.end(), [&](int a, int b) { return ucost(a) > ucost(b); });
  std::vector<long long> wload(WR, 0);
  std::vector<int> wcount(WR, 0);
  std::vector<int> slot_group(NS, -1);
  for (int u : uorder) {
    int bw = -1;
    for (int w = 0; w < WR; ++w)
      if (wcount[w] + gu <= NIT && (bw < 0 || wload[w] < wload[bw])) bw = w;
    FR_REQUIRE(bw >= 0, "panel_op_build: slot assignment failed");
    for (int j = 0; j < gu; ++j) slot_group[bw * NIT + wcount[bw] + j] = u * gu + j;
    wcount[bw] += gu;
    wload[bw] += ucost(u);
  }
  // ---- pack
  std::vector<T> vals;
  std::vector<uint32_t> idx;
  std::vector<int> off(nchunks * NS + 1, 0);
  std::vector<int> rowmap(NS * 8, -1);
  for (int s = 0; s < NS; ++s)
    if (slot_group[s] >= 0)
      for (int r = 0; r < 8; ++r) {
        const int m = order[8 * slot_group[s] + r];
        rowmap[s * 8 + r] = (m >= 0 && opt.row_ids) ? opt.row_ids[m] : m;
      }
  long long macs = 0;
  int nblk = 0;
  if (!sparse) {
    // dense: blocks ordered (chunk, k-block, slot); rows of a block are the consecutive stage rows 4b..4b+3 (FP64) / row b (FP32)
    for (int c = 0; c < nchunks; ++c) {
      chunks[c].base = nblk / NS;
      const int n = (int)chunk_cols[c].size();
      const int nb = f64 ? (n + 3) / 4 : n;
      for (int b = 0; b < nb; ++b)
        for (int s = 0; s < NS; ++s) {
          const int g = slot_group[s];
          if (f64) {
            for (int lane = 0; lane < 32; ++lane) {
              const int r = lane >> 2, j = lane & 3;
              const int m = g >= 0 ? order[8 * g + r] : -1;
              vals.push_back((T)((m >= 0 && 4 * b + j < n) ? A[(size_t)m * K + chunk_cols[c][4 * b + j]] : 0.0));
            }
            if (g >= 0) macs += 32;
          } else {
            for (int r = 0; r < 8; ++r) {
              const int m = g >= 0 ? order[8 * g + r] : -1;
              vals.push_back((T)(m >= 0 ? A[(size_t)m * K + chunk_cols[c][b]] : 0.0));
            }
            if (g >= 0) macs += 8;
          }
          ++nblk;
        }
    }
  }
  for (int c = 0; c < nchunks && sparse; ++c)
    for (int s = 0; s < NS; ++s) {
      off[c * NS + s] = nblk;
      const int g = slot_group[s];
      if (g < 0) continue;
      const std::vector<int> &L = lists[g][c];
      const int n = (int)L.size();
      if (f64) {
        for (int b = 0; b < (n + 3) / 4; ++b) {
          for (int j = 0; j < 4; ++j) {
            const int kk = 4 * b + j < n ? L[4 * b + j] : 0;
            idx.push_back((uint32_t)kk * (uint32_t)(PV * geo.NE + 4) * (uint32_t)sizeof(T));
          }
          for (int lane = 0; lane < 32; ++lane) {
            const int r = lane >> 2, j = lane & 3;
            const int m = order[8 * g + r];
            double v = 0;
            if (m >= 0 && 4 * b + j < n) v = A[(size_t)m * K + chunk_cols[c][L[4 * b + j]]];
            if (sparse && std::fabs(v) <= thr) v = 0;
            vals.push_back((T)v);
          }
          ++nblk;
          macs += 32;
        }
      } else {
        for (int b = 0; b < n; ++b) {
          idx.push_back((uint32_t)L[b] * (uint32_t)(PV * geo.NE + 4) * (uint32_t)sizeof(T));
          for (int r = 0; r < 8; ++r) {
            const int m = order[8 * g + r];
            double v = m >= 0 ? A[(size_t)m * K + chunk_cols[c][L[b]]] : 0.0;
            if (sparse && std::fabs(v) <= thr) v = 0;
            vals.push_back((T)v);
          }
          ++nblk;
          macs += 8;
        }
      }
    }
  if (sparse) off[nchunks * NS] = nblk;
  // the multiply loop prefetches two blocks ahead: two all-zero blocks close the arrays (not counted in nblk)
  for (int d = 0; d < 2; ++d) {
    for (int j = 0; j < (f64 ? 4 : 1); ++j) idx.push_back(0u);
    for (int j = 0; j < (f64 ? 32 : 8); ++j) vals.push_back(T(0));
  }
  const size_t smem_op = ((vals.size() * sizeof(T) + 15) / 16 * 16) + ((idx.size() * 4 + 15) / 16 * 16) +
                         ((off.size() * 4 + 15) / 16 * 16) + ((rowmap.size() * 4 + 15) / 16 * 16) +
                         ((chunks.size() * sizeof(ChunkDesc) + 15) / 16 * 16);
  if (geo.occ == 2) smem_total = smem_total / 2 - 2048;
  if (smem_op > smem_budget || smem_op + 8192 > smem_total) return false;
  size_t stage_elems = 0;
  const int LDBh = PV * geo.NE + 4;
  for (auto &c : chunks)
    stage_elems = std::max(stage_elems, c.kind == KIND_FLUX ? flux_stage_elems(c.nrows, geo.NE, LDBh, opt.curved) : (size_t)c.nrows * LDBh);
  if (smem_op + (size_t)geo.NG * PANEL_NSTAGE * stage_elems * sizeof(T) + 16 > smem_total) {
    // MAC rows per chunk that would fit: scale the tallest chunk down proportionally (flux chunks carry 4/3 rows + metrics)
    if (smem_total > smem_op + 4096) {
      const double room = (double)(smem_total - smem_op - 1024) / ((double)PANEL_NSTAGE * geo.NG * sizeof(T));
      *kc_fit = (int)(kcmax * room / (double)stage_elems);
    }
    return false;
  }
  panel_op_free(p);
  p.M = M;
  p.K = K;
  p.WR = WR;
  p.WC = geo.WC;
  p.NIT = NIT;
  p.CX = geo.CX;
  p.NE = geo.NE;
  p.NG = geo.NG;
  p.occ = geo.occ;
  p.KC = kcmax;
  p.stage_elems = (int)stage_elems;
  p.curved = opt.curved;
  p.nchunks = nchunks;
  p.NS = NS;
  p.nblk = nblk;
  p.nidx = (int)idx.size();
  p.dbg = getenv("FRB_PANEL_DBG") ? atoi(getenv("FRB_PANEL_DBG")) : 0;
  if (getenv("FRB_PANEL_VERBOSE"))
    fprintf(stderr, "panel_op %s M=%d K=%d %s G=%d WR=%d WC=%d NIT=%d CX=%d NE=%d NG=%d occ=%d warps=%d KC=%d nchunks=%d nblk=%d smem_op=%zu stage=%zu B density=%.2f macs/col=%.0f (dense %d)\n",
            f64 ? "f64" : "f32", M, K, sparse ? "sparse" : "dense", G, WR, geo.WC, NIT, geo.CX, geo.NE, geo.NG, geo.occ, geo.NG * WR * geo.WC, kcmax,
            nchunks, nblk, smem_op, stage_elems * sizeof(T), density, (double)macs, M * K);
  p.sparse = sparse ? 1 : 0;
  p.macs_per_col = (double)macs;
  p.density = density;
  p.smem_op = smem_op;
  auto up = [](auto *&dst, const auto &h) {
    using E = typename std::remove_reference<decltype(h[0])>::type;
    const size_t nb = std::max<size_t>(h.size(), 1) * sizeof(E);
    FR_CUDA_TRY(cudaMalloc((void **)&dst, nb));
    if (!h.empty()) FR_CUDA_TRY(cudaMemcpy((void *)dst, h.data(), h.size() * sizeof(E), cudaMemcpyHostToDevice));
  };
  up(p.vals, vals);
  up(p.idx, idx);
  up(p.off, off);
  up(p.rowmap, rowmap);
  up(p.chunks, chunks);
  return true;
}

// ------------------------------------------------------------------------------------------------ device side
#ifdef __CUDACC__

__device__ __forceinline__ void pcp_async16(void *smem, const void *gmem, int src_bytes) {
  unsigned s = (unsigned)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(s), "l"(gmem), "r"(src_bytes));
}
__device__ __forceinline__ void prefetch_l2(const void *p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }
__device__ __forceinline__ void pcp_commit() { asm volatile("cp.async.commit_group;\n" ::); }
template <int N>
__device__ __forceinline__ void pcp_wait() {
  asm volatile("cp.async.wait_group %0;\n" ::"n"(N));
}

__device__ __forceinline__ void dmma884(double &c0, double &c1, double a, double b) {
  asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
               : "+d"(c0), "+d"(c1)
               : "d"(a), "d"(b));
}

// Shared-memory view of the packed operator.
template <typename T>
struct OpSmem {
  const T *vals;
  const uint32_t *idx;
  const int *off;
  const int *rowmap;
  const ChunkDesc *chunks;
};

template <typename T>
__device__ __forceinline__ char *op_smem_carve(char *base, const PanelOp<T> &op, OpSmem<T> &v) {
  auto al = [](size_t n) { return (n + 15) / 16 * 16; };
  const size_t nv = (size_t)(op.nblk + 2) * (sizeof(T) == 8 ? 32 : 8) * sizeof(T);
  v.vals = reinterpret_cast<const T *>(base);
  base += al(nv);
  v.idx = reinterpret_cast<const uint32_t *>(base);
  base += al((size_t)op.nidx * 4);
  v.off = reinterpret_cast<const int *>(base);
  base += al(((size_t)op.nchunks * op.NS + 1) * 4);
  v.rowmap = reinterpret_cast<const int *>(base);
  base += al((size_t)op.NS * 8 * 4);
  v.chunks = reinterpret_cast<const ChunkDesc *>(base);
  base += al((size_t)op.nchunks * sizeof(ChunkDesc));
  return base;
}

// Copy the operator image global -> shared with cp.async (all threads), one commit group.
template <typename T>
__device__ __forceinline__ void op_smem_load(char *base, const PanelOp<T> &op, int tid, int nthreads) {
  auto al = [](size_t n) { return (n + 15) / 16 * 16; };
  auto copy = [&](char *dst, const void *src, size_t nbytes) {
    const int np = (int)(al(nbytes) / 16);
    for (int p = tid; p < np; p += nthreads) {
      const int rem = (int)nbytes - 16 * p;
      pcp_async16(dst + 16 * p, reinterpret_cast<const char *>(src) + 16 * p, rem >= 16 ? 16 : rem);
    }
    return dst + al(nbytes);
  };
  char *b = base;
  b = copy(b, op.vals, (size_t)(op.nblk + 2) * (sizeof(T) == 8 ? 32 : 8) * sizeof(T));
  b = copy(b, op.idx, (size_t)op.nidx * 4);
  b = copy(b, op.off, ((size_t)op.nchunks * op.NS + 1) * 4);
  b = copy(b, op.rowmap, (size_t)op.NS * 8 * 4);
  b = copy(b, op.chunks, (size_t)op.nchunks * sizeof(ChunkDesc));
}

// ---- accumulators and the multiply-accumulate core.  Panel columns in shared memory: c = v*NE + e, row pitch LDB.
template <typename T, int NIT, int CX>
struct Acc;

// FP64: per slot, CX column blocks of 8 elements x 5 variables, one m8n8k4 C fragment (2 doubles) each.
template <int NIT, int CX>
struct Acc<double, NIT, CX> {
  double c[NIT][CX][PV][2];
  __device__ __forceinline__ void zero() {
#pragma unroll
    for (int i = 0; i < NIT; ++i)
#pragma unroll
      for (int b = 0; b < CX; ++b)
#pragma unroll
        for (int v = 0; v < PV; ++v) c[i][b][v][0] = c[i][b][v][1] = 0.0;
  }
  // elements of the panel this warp-column owns: [wc*8*CX, (wc+1)*8*CX)
  __device__ __forceinline__ void mac_chunk(const OpSmem<double> &A, int chunk, int NS, int slot0, const double *Bst, int LDB,
                                            int NE, int wc, int lane) {
    // 32-bit byte-offset arithmetic inside the shared window.  The warp's blocks of this chunk are contiguous across
    // its NIT slots, so one software pipeline runs through all of them: operator value and row offset are fetched two
    // blocks ahead, the B fragments one block ahead of the DMMAs that consume them.
    const char *bcol = reinterpret_cast<const char *>(Bst + wc * 8 * CX + (lane >> 2));
    const char *av = reinterpret_cast<const char *>(A.vals) + lane * 8;
    const char *ai = reinterpret_cast<const char *>(A.idx) + (lane & 3) * 4;
    const uint32_t vs = (uint32_t)NE * 8u;
    const int *offp = A.off + chunk * NS + slot0;
    int b = offp[0];
    double a0 = *reinterpret_cast<const double *>(av + (uint32_t)b * 256u);
    double a1 = *reinterpret_cast<const double *>(av + (uint32_t)b * 256u + 256u);
    uint32_t ro1 = *reinterpret_cast<const uint32_t *>(ai + (uint32_t)b * 16u + 16u);
    double bf0[PV][CX];
    {
      const char *bp = bcol + *reinterpret_cast<const uint32_t *>(ai + (uint32_t)b * 16u);
#pragma unroll
      for (int v = 0; v < PV; ++v) {
#pragma unroll
        for (int cb = 0; cb < CX; ++cb) bf0[v][cb] = *reinterpret_cast<const double *>(bp + cb * 64);
        bp += vs;
      }
    }
#pragma unroll
    for (int i = 0; i < NIT; ++i) {
      const int bend = offp[i + 1];
#pragma unroll 2
      for (; b < bend; ++b) {
        double bf1[PV][CX];
        const char *bp = bcol + ro1;
#pragma unroll
        for (int v = 0; v < PV; ++v) {
#pragma unroll
          for (int cb = 0; cb < CX; ++cb) bf1[v][cb] = *reinterpret_cast<const double *>(bp + cb * 64);
          bp += vs;
        }
        const double a2 = *reinterpret_cast<const double *>(av + (uint32_t)b * 256u + 512u);
        const uint32_t ro2 = *reinterpret_cast<const uint32_t *>(ai + (uint32_t)b * 16u + 32u);
#pragma unroll
        for (int v = 0; v < PV; ++v)
#pragma unroll
          for (int cb = 0; cb < CX; ++cb) dmma884(c[i][cb][v][0], c[i][cb][v][1], a0, bf0[v][cb]);
        a0 = a1;
        a1 = a2;
        ro1 = ro2;
#pragma unroll
        for (int v = 0; v < PV; ++v)
#pragma unroll
          for (int cb = 0; cb < CX; ++cb) bf0[v][cb] = bf1[v][cb];
      }
    }
  }
  // Dense operator: the NIT row groups of the warp share the chunk's rows, so the B fragments of a k-block (stage rows
  // 4b..4b+3) are loaded once and feed NIT x 5 x CX DMMAs; no index list.
  __device__ __forceinline__ void mac_dense(const OpSmem<double> &A, const ChunkDesc &cd, int NS, int slot0, const double *Bst,
                                            int LDB, int NE, int wc, int lane) {
    const char *bcol = reinterpret_cast<const char *>(Bst + wc * 8 * CX + (lane >> 2));
    const char *av = reinterpret_cast<const char *>(A.vals) + ((uint32_t)(cd.base * NS + slot0) * 32u + lane) * 8u;
    const uint32_t vs = (uint32_t)NE * 8u, rs = (uint32_t)LDB * 8u, as = (uint32_t)NS * 256u;
    const int nb = (cd.nrows + 3) >> 2, last = cd.nrows - 1;
    const int kl = lane & 3;
#pragma unroll 2
    for (int b = 0; b < nb; ++b) {
      const int row = min(4 * b + kl, last);           // padded rows of the last block: operator is zero, data must be finite
      const char *bp = bcol + (uint32_t)row * rs;
      double bf[PV][CX];
#pragma unroll
      for (int v = 0; v < PV; ++v) {
#pragma unroll
        for (int cb = 0; cb < CX; ++cb) bf[v][cb] = *reinterpret_cast<const double *>(bp + cb * 64);
        bp += vs;
      }
      const char *ap = av + (uint32_t)b * as;
#pragma unroll
      for (int i = 0; i < NIT; ++i) {
        const double a = *reinterpret_cast<const double *>(ap + i * 256);
#pragma unroll
        for (int v = 0; v < PV; ++v)
#pragma unroll
          for (int cb = 0; cb < CX; ++cb) dmma884(c[i][cb][v][0], c[i][cb][v][1], a, bf[v][cb]);
      }
    }
  }
  // f(i, rr, e, tile[PV][EW]): slot i, thread-local row rr, first element e of EW consecutive ones, all 5 variables
  template <typename F>
  __device__ __forceinline__ void foreach_tile(int wc, int lane, F &&f) {
#pragma unroll
    for (int i = 0; i < NIT; ++i)
#pragma unroll
      for (int cb = 0; cb < CX; ++cb) f(i, 0, wc * 8 * CX + cb * 8 + 2 * (lane & 3), c[i][cb]);
  }
  // f(i, rr, e): coordinates only (for prefetching what the epilogue will read)
  template <typename F>
  __device__ __forceinline__ void foreach_coord(int wc, int lane, F &&f) {
#pragma unroll
    for (int i = 0; i < NIT; ++i)
#pragma unroll
      for (int cb = 0; cb < CX; ++cb) f(i, 0, wc * 8 * CX + cb * 8 + 2 * (lane & 3));
  }
  // f(t, rr, e, tile_a0, tile_a1, tile_a2): slots 3t, 3t+1, 3t+2 hold the three alpha of the same rows
  template <typename F>
  __device__ __forceinline__ void foreach_triple(int wc, int lane, F &&f) {
#pragma unroll
    for (int t = 0; t < NIT / 3; ++t)
#pragma unroll
      for (int cb = 0; cb < CX; ++cb)
        f(t, 0, wc * 8 * CX + cb * 8 + 2 * (lane & 3), c[3 * t][cb], c[3 * t + 1][cb], c[3 * t + 2][cb]);
  }
  // g(i, rr, r): thread-local row index rr of slot i is row r of the 8-row group
  template <typename G>
  __device__ __forceinline__ void foreach_row(int lane, G &&g) {
#pragma unroll
    for (int i = 0; i < NIT; ++i) g(i, 0, lane >> 2);
  }
  static constexpr int EW = 2;   // consecutive elements per foreach2 call
  static constexpr int ROWS = 1; // rows per thread per slot
  static constexpr int NSLOT = NIT;
};

// FP32: per slot, 8 rows x 5 variables x CX elements per lane.
template <int NIT, int CX>
struct Acc<float, NIT, CX> {
  float c[NIT][8][PV][CX];
  __device__ __forceinline__ void zero() {
#pragma unroll
    for (int i = 0; i < NIT; ++i)
#pragma unroll
      for (int r = 0; r < 8; ++r)
#pragma unroll
        for (int v = 0; v < PV; ++v)
#pragma unroll
          for (int j = 0; j < CX; ++j) c[i][r][v][j] = 0.f;
  }
  __device__ __forceinline__ void mac_chunk(const OpSmem<float> &A, int chunk, int NS, int slot0, const float *Bst, int LDB,
                                            int NE, int wc, int lane) {
    const char *bcol = reinterpret_cast<const char *>(Bst + wc * 32 * CX + lane * CX);
    const char *avp = reinterpret_cast<const char *>(A.vals);
    const uint32_t vs = (uint32_t)NE * 4u;
#pragma unroll
    for (int i = 0; i < NIT; ++i) {
      const int b0 = A.off[chunk * NS + slot0 + i], b1 = A.off[chunk * NS + slot0 + i + 1];
#pragma unroll 2
      for (int b = b0; b < b1; ++b) {
        const float4 a0 = *reinterpret_cast<const float4 *>(avp + (uint32_t)b * 32u);
        const float4 a1 = *reinterpret_cast<const float4 *>(avp + (uint32_t)b * 32u + 16u);
        const float av[8] = {a0.x, a0.y, a0.z, a0.w, a1.x, a1.y, a1.z, a1.w};
        const char *bp = bcol + A.idx[b];
        float bv[PV][CX];
#pragma unroll
        for (int v = 0; v < PV; ++v) {
          if (CX == 2) {
            const float2 t = *reinterpret_cast<const float2 *>(bp);
            bv[v][0] = t.x;
            bv[v][CX - 1] = t.y;
          } else {
            bv[v][0] = *reinterpret_cast<const float *>(bp);
          }
          bp += vs;
        }
#pragma unroll
        for (int r = 0; r < 8; ++r)
#pragma unroll
          for (int v = 0; v < PV; ++v)
#pragma unroll
            for (int j = 0; j < CX; ++j) c[i][r][v][j] = fmaf(av[r], bv[v][j], c[i][r][v][j]);
      }
    }
  }
  // Dense operator: one B row feeds the NIT row groups of the warp.
  __device__ __forceinline__ void mac_dense(const OpSmem<float> &A, const ChunkDesc &cd, int NS, int slot0, const float *Bst,
                                            int LDB, int NE, int wc, int lane) {
    const char *bp0 = reinterpret_cast<const char *>(Bst + wc * 32 * CX + lane * CX);
    const char *ap0 = reinterpret_cast<const char *>(A.vals) + (uint32_t)(cd.base * NS + slot0) * 32u;
    const uint32_t vs = (uint32_t)NE * 4u, rs = (uint32_t)LDB * 4u, as = (uint32_t)NS * 32u;
#pragma unroll 2
    for (int k = 0; k < cd.nrows; ++k) {
      const char *bp = bp0 + (uint32_t)k * rs;
      float bv[PV][CX];
#pragma unroll
      for (int v = 0; v < PV; ++v) {
        if (CX == 2) {
          const float2 t = *reinterpret_cast<const float2 *>(bp);
          bv[v][0] = t.x;
          bv[v][CX - 1] = t.y;
        } else {
          bv[v][0] = *reinterpret_cast<const float *>(bp);
        }
        bp += vs;
      }
      const char *ap = ap0 + (uint32_t)k * as;
#pragma unroll
      for (int i = 0; i < NIT; ++i) {
        const float4 a0 = *reinterpret_cast<const float4 *>(ap + i * 32);
        const float4 a1 = *reinterpret_cast<const float4 *>(ap + i * 32 + 16);
        const float av[8] = {a0.x, a0.y, a0.z, a0.w, a1.x, a1.y, a1.z, a1.w};
#pragma unroll
        for (int r = 0; r < 8; ++r)
#pragma unroll
          for (int v = 0; v < PV; ++v)
#pragma unroll
            for (int j = 0; j < CX; ++j) c[i][r][v][j] = fmaf(av[r], bv[v][j], c[i][r][v][j]);
      }
    }
  }
  template <typename F>
  __device__ __forceinline__ void foreach_tile(int wc, int lane, F &&f) {
#pragma unroll
    for (int i = 0; i < NIT; ++i)
#pragma unroll
      for (int r = 0; r < 8; ++r) f(i, r, wc * 32 * CX + lane * CX, c[i][r]);
  }
  template <typename F>
  __device__ __forceinline__ void foreach_coord(int wc, int lane, F &&f) {
#pragma unroll
    for (int i = 0; i < NIT; ++i)
#pragma unroll
      for (int r = 0; r < 8; ++r) f(i, r, wc * 32 * CX + lane * CX);
  }
  template <typename F>
  __device__ __forceinline__ void foreach_triple(int wc, int lane, F &&f) {
#pragma unroll
    for (int t = 0; t < NIT / 3; ++t)
#pragma unroll
      for (int r = 0; r < 8; ++r) f(t, r, wc * 32 * CX + lane * CX, c[3 * t][r], c[3 * t + 1][r], c[3 * t + 2][r]);
  }
  template <typename G>
  __device__ __forceinline__ void foreach_row(int lane, G &&g) {
#pragma unroll
    for (int i = 0; i < NIT; ++i)
#pragma unroll
      for (int r = 0; r < 8; ++r) g(i, r, r);
  }
  static constexpr int EW = CX;
  static constexpr int ROWS = 8;
  static constexpr int NSLOT = NIT;
};

#endif  // __CUDACC__

}  // namespace frb
