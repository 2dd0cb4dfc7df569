// Panel kernels: the operator products C <- c1*A*B + c2*C (eq. 1) and their fusions with the adjacent
// point-wise work, for one element type.  "A is a constant operator matrix, and B and C are row-major state matrices"
// (PAPER.md:39): every column of B is independent, so one CTA owns a *panel* of NE consecutive elements (all 5
// conserved variables = 5*NE columns) and ALL rows of A -- the column slicing the paper's OpenMP backend found best
// -- while B streams through shared memory in K-chunks and the accumulators stay in registers.
//
// B200 design:
//   * the operator is packed once at fr_setup into 8-row groups (dense operators: every k of a chunk, in k-blocks shared by
//     all groups; sparse operators: per group a compact list of the k that are non-zero in it) and stays resident in shared
//     memory for the life of the persistent CTA (plain products whose image exceeds shared memory stream the packed blocks
//     through the ring instead: PanelOp::streamed);
//   * B chunks are moved by the TMA unit (cp.async.bulk.tensor from tensor maps over the state matrices, tma.cuh): a producer
//     warp per warp group issues the copies into a ring of stages, each stage guarded by a full and an empty mbarrier; the
//     consumer warps never issue a copy and never meet at a CTA-wide barrier;
//   * FP64 multiplies on the FP64 tensor pipe, mma.sync.m8n8k4.f64 (DMMA), reading its B fragments from the 128-byte-swizzled
//     stage; the four rows of a k-block are chosen at set-up so that these loads are bank-conflict free;
//     FP32 multiplies on register tiles of 8 rows x 5 variables x (1|2) elements with packed fma.rn.f32x2 (two IEEE FP32 FMAs per
//     instruction; the gradient kernels keep scalar FFMA) -- no TF32: the 2e-5 parity bound excludes it, and tcgen05 has no FP32/FP64 kind;
//   * the chunking of K and the composition of every k-block depend on the operator alone, never on the launch geometry, so
//     every geometry the autotuner may pick gives bit-identical results;
//   * epilogues (what happens to the accumulators) are policies, which is how the gradient transform, the -1/|J| scaling and
//     the Runge-Kutta stage update are fused into the products.
#pragma once
#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <numeric>

#include "common.cuh"

namespace frb {

constexpr int PV = FR_NVAR;          // variable segments per panel
constexpr int PANEL_MAXW = 20;       // warps per CTA, producers included (fewer when the accumulators need more registers)
constexpr int PANEL_MAXCHUNKS = 160;
constexpr int PANEL_KCMAX = 40;      // rows per chunk (upper bound; a multiple of 8)
constexpr int PANEL_MAXSTAGE = 8;    // ring depth (upper bound)
constexpr int PANEL_MAXSRC = 2;      // matrices stacked along K

// One K-chunk of the stacked right-hand operand: rows [row0, row0+nrows) of source `src`, copied as a box of `step` rows.
struct ChunkDesc {
  int src, row0, nrows, step;
  int base, nblk, pad0, pad1;   // dense operators: first packed block of this chunk and their number (FP64: k-blocks of 4 rows; FP32: rows)
};

// Device image of a packed operator + its launch geometry (all pointers device).
template <typename T>
struct PanelOp {
  int M = 0, K = 0;
  int WR = 0, WC = 0, NIT = 0, CX = 0;   // warp grid, row groups per row-warp, column blocks (FP64) / elements per lane (FP32)
  int NE = 0;                            // elements per panel (of one warp group)
  int NG = 1;                            // independent warp groups per CTA, each streaming its own panels (staggered)
  int occ = 1;                           // CTAs per SM the plan was sized for (shared memory and registers)
  int nchunks = 0, NS = 0;               // chunks, slots = WR*NIT
  int nstage = 0;                        // ring depth
  int stage_bytes = 0;                   // bytes of one ring stage (multiple of 1024)
  int nblk = 0;                          // packed blocks (FP64: 8x4 tiles; FP32: 8x1 columns)
  int nidx = 0;                          // entries of idx
  int pf_epi = 0;                        // the epilogue's global operands are pulled into L2 before the last chunk (set by the launcher)
#ifdef FRB_DEBUG_KNOBS
  int dbg = 0;                           // measurement aid (env FRB_PANEL_DBG): 1 skip multiply, 2 skip epilogue
#endif
  int sparse = 0;                        // 1: per-group k-lists (idx/off); 0: dense, all slots share the chunk's k-blocks
  int nsrc = 0;
  int src_rows[PANEL_MAXSRC] = {0, 0};   // rows of each stacked source
  int src_step[PANEL_MAXSRC] = {0, 0};   // rows per chunk (TMA box height) of each source
  double macs_per_col = 0;               // executed multiply-adds per column (dense: M*K)
  double density = 1;                    // fraction of non-zero entries of the operator
  T *vals = nullptr;                     // FP64 [nblk][32]; FP32 [nblk][8]
  uint32_t *idx = nullptr;               // byte offset of the B row in a stage plane: FP64 [..][4] (swizzle term included), FP32 [..]
  int *off = nullptr;                    // sparse: [nchunks*NS + 1]
  int *rowmap = nullptr;                 // [NS*8] actual row of (slot, r) or -1
  ChunkDesc *chunks = nullptr;           // [nchunks]
  size_t smem_op = 0;                    // bytes of the operator image in shared memory
  size_t bytes_vals = 0, bytes_idx = 0, bytes_off = 0, bytes_rowmap = 0, bytes_chunks = 0;   // each a multiple of 16
  bool ok() const { return vals != nullptr; }
  // Streamed operator (plain products whose image exceeds shared memory): the packed blocks do not stay in shared memory
  // (bytes_vals = 0) but travel through the ring behind each chunk's rows of B (dense packing, one source), at stage offset a_off().
  __host__ __device__ bool streamed() const { return vals != nullptr && bytes_vals == 0; }
  __host__ __device__ int a_off() const { return (PV * NE * src_step[0] * (int)sizeof(T) + 127) / 128 * 128; }
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

// How the K dimension of the operator is fed: a list of matrices stacked along K, `rows` plain rows each <-> `rows` columns of A.
struct KSource {
  int rows;
};

struct PanelGeom {
  int WR, WC, NIT, CX, NE;
  double eff;
  int NG;
  int occ;
};

// Warps per CTA (consumers + one producer per group) a given accumulator shape allows: a multiple of four (ptxas sizes the
// register budget for whole quads of warps, one per SM sub-partition), the largest whose register share still leaves the
// accumulators 68 registers of head-room (less spills loop-carried scalars, which costs a local-memory round trip per chunk).  FP64: NIT*CX*10 doubles per thread; FP32: NIT*CX*40 floats.
template <typename T>
constexpr int panel_maxw(int nit, int cx, bool triple = false) {
  // FP32 tiles also keep 8 operator values and 5*CX state values live per k and index more arrays: the CX = 2 shapes spill
  // inside the multiply loop with little head-room (8x slower), so FP32 with CX = 2 budgets +110.
  const int need = (sizeof(T) == 8 ? nit * cx * 20 : nit * cx * 40) + ((sizeof(T) == 4 && cx == 2) ? 110 : 68);
  // the gradient operators of prisms (10 triples of row groups) need 10 row-warps of NIT = 6 (FP64) / NIT = 3 (FP32): in the
  // gradient kernels these two shapes take 12 warps at 168 registers and spill ~150 bytes in the epilogue
  if (triple && (sizeof(T) == 8 ? nit * cx == 6 : nit * cx == 3)) return 12;
  int w = PANEL_MAXW / 4 * 4;
  while (w > 8 && 2048 / w < need) w -= 4;
  return w;
}

// Candidate launch geometries for G row groups, best static score first.  The FP64 tensor pipe is per SM sub-partition: the
// multiplying warps should spread evenly over the four of them.
template <typename T>
inline std::vector<PanelGeom> list_geoms(int G, int min_ne, int max_ne, int triple, bool dense) {
  std::vector<PanelGeom> all;
  const bool f64 = sizeof(T) == 8;
  const int gu = triple ? 3 : 1;            // groups come in units of `gu` that must stay on one row-warp
  const int GU = (G + gu - 1) / gu;
  const int ngmax = getenv("FRB_PANEL_NG") ? atoi(getenv("FRB_PANEL_NG")) : 2;
  for (int NG = 1; NG <= ngmax; ++NG)
    for (int WR = 1; WR <= PANEL_MAXW; ++WR) {
      const int nit = ((GU + WR - 1) / WR) * gu;
      if (WR > 1 && ((GU + WR - 2) / (WR - 1)) * gu == nit) continue;   // same accumulators with fewer row-warps exist: skip the idle ones
      for (int WC = 1; NG * WR * WC + NG <= PANEL_MAXW; ++WC) {
        for (int CX = 2; CX >= 1; --CX) {
          if (f64 ? nit * CX > 8 : nit * CX > 4) continue;
          const int W = NG * WR * WC;                          // consumer warps
          if (W + NG > panel_maxw<T>(nit, CX, triple != 0)) continue;
          const int NE = (f64 ? 8 : 32) * CX * WC;
          // panels tile the padded leading dimension (a multiple of 128) exactly; FP64 stages are made of 16-element blocks
          if (NE < min_ne || NE > max_ne || 128 % NE != 0 || (f64 && NE % 16)) continue;
          const double eff = (double)G / (WR * nit);
          // spread over the sub-partitions: the busiest of the four bounds the multiply rate
          const double bal = (double)W / (4.0 * ((W + 3) / 4));
          double score = eff * bal * (0.4 + 0.6 * std::min(W, 12) / 12.0) * (1.0 + 0.02 * std::log2((double)NE)) * (1.0 - 0.005 * nit * CX);
          // dense operators: the B fragments of a k-block are shared by the NIT row groups of the warp
          if (dense) score /= 1.0 + 0.4 * (2.0 / nit + 0.4 / CX);
          // two staggered warp groups hide one group's epilogue behind the other's multiplies
          if (NG == 2) score *= f64 ? 1.15 : 0.9;
          all.push_back(PanelGeom{WR, WC, nit, CX, NE, score, NG, 1});
          // two CTAs per SM (half the shared memory and registers each): the other way to overlap one panel's epilogue with
          // another's multiplies; only timing (fr_setup autotuning) tells which wins
          if (NG == 1 && 2 * (W + 1) <= panel_maxw<T>(nit, CX, triple != 0)) all.push_back(PanelGeom{WR, WC, nit, CX, NE, score * 0.9, NG, 2});
        }
      }
    }
  std::stable_sort(all.begin(), all.end(), [](const PanelGeom &x, const PanelGeom &y) { return x.eff > y.eff; });
  return all;
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
  int allow_sparse = 1;
  int cand = 0;            // k-th best geometry by static score (autotuning)
  const int *row_ids = nullptr;   // row split: the epilogue's row number of each row of A (nullptr = 0..M-1)
  // entries with |a| <= drop_rel * max|A| are treated as structural zeros (reading R24); 0: only exact zeros
  double drop_rel = 1.4210854715202004e-14;
  int stream = 0;          // build the streamed-operator form (PanelOp::stream)
};

// Rows per chunk of a source with `rows` rows: the multiple of 8 (<= PANEL_KCMAX) with the fewest chunks, counting a fixed
// per-chunk overhead worth six rows.  A function of `rows` alone (see the determinism note at the top).
inline int panel_chunk_step(int rows, int cap = PANEL_KCMAX) {
  int best = 8;
  long bestc = 1l << 60;
  for (int step = 8; step <= cap; step += 8) {
    const long nch = (rows + step - 1) / step;
    const long c = nch * (step + 6);
    if (c <= bestc) {
      bestc = c;
      best = step;
    }
  }
  return best;
}

// The four stage rows of each k-block of a chunk with n rows (FP64).  Inside a group of eight consecutive rows the even and
// the odd rows form one block each: with the 128-byte swizzle the rows of a block then differ in (row & 7) >> 1, which makes
// the DMMA B-fragment loads bank-conflict free.  A tail of at most four rows is one block.
inline std::vector<std::vector<int>> dense_blocks_f64(int n) {
  std::vector<std::vector<int>> out;
  for (int g = 0; g < n; g += 8) {
    const int t = std::min(8, n - g);
    if (t <= 4) {
      std::vector<int> b;
      for (int j = 0; j < t; ++j) b.push_back(g + j);
      out.push_back(b);
    } else {
      std::vector<int> ev, od;
      for (int j = 0; j < t; ++j) (j & 1 ? od : ev).push_back(g + j);
      out.push_back(ev);
      out.push_back(od);
    }
  }
  return out;
}

// Blocks of four from a list of stage rows, rows of a block from different bank classes ((row & 7) >> 1) where possible.
inline std::vector<std::vector<int>> sparse_blocks_f64(const std::vector<int> &rows) {
  std::vector<std::vector<int>> bucket(4), out;
  for (int r : rows) bucket[(r & 7) >> 1].push_back(r);
  size_t pos[4] = {0, 0, 0, 0};
  size_t left = rows.size();
  while (left > 0) {
    std::vector<int> b;
    bool took[4] = {false, false, false, false};
    while (b.size() < 4 && left > 0) {
      // the fullest class not yet in this block; when every class with rows left is in it already, the fullest one again
      int q = -1;
      for (int pass = 0; pass < 2 && q < 0; ++pass)
        for (int c = 0; c < 4; ++c) {
          const size_t rem = bucket[c].size() - pos[c];
          if (rem == 0 || (pass == 0 && took[c])) continue;
          if (q < 0 || rem > bucket[q].size() - pos[q]) q = c;
        }
      b.push_back(bucket[q][pos[q]++]);
      took[q] = true;
      --left;
    }
    out.push_back(b);
  }
  return out;
}

// byte offset of stage row r inside a plane, with the swizzle term of its 128-byte line in bits 4..6
inline uint32_t swz_row_offset(int r) { return (uint32_t)r * 128u + (uint32_t)(r & 7) * 16u; }

// Pack A (M x K, host FP64, row-major) for the panel kernels.  `srcs` stacks the K dimension.  Returns false if the
// operator does not fit the resident-in-shared-memory design with geometry candidate opt.cand (or the candidate does not exist).
template <typename T>
bool panel_op_build(PanelOp<T> &p, int M, int K, const double *A, const std::vector<KSource> &srcs, const PackOptions &opt_in,
                    size_t smem_budget, size_t smem_total_in = 226 * 1024) {
  PackOptions opt = opt_in;
  // FRB_FORCE_CAND=k: build geometry candidate k where the caller asked for the default; falls back to the default if k does
  // not exist for this operator.  Lets the parity tests cover every candidate the autotuner may pick.
  if (opt.cand == 0 && getenv("FRB_FORCE_CAND")) {
    PackOptions o2 = opt;
    o2.cand = atoi(getenv("FRB_FORCE_CAND"));
    if (o2.cand > 0 && panel_op_build(p, M, K, A, srcs, o2, smem_budget, smem_total_in)) return true;
  }
  const bool f64 = sizeof(T) == 8;
  FR_REQUIRE((int)srcs.size() >= 1 && (int)srcs.size() <= PANEL_MAXSRC, "panel_op_build: one or two stacked sources");
  int ktot = 0;
  for (auto &s : srcs) ktot += s.rows;
  FR_REQUIRE(ktot == K, "panel_op_build: sources do not add up to K");
  double amax = 0;
  for (size_t i = 0; i < (size_t)M * K; ++i) {
    FR_REQUIRE(A[i] == A[i] && A[i] - A[i] == 0.0, "operator contains non-finite entries");
    amax = std::max(amax, std::fabs(A[i]));
  }
  const double thr = amax * opt.drop_rel;
  std::vector<std::vector<uint8_t>> sup(M, std::vector<uint8_t>(K, 0));
  size_t nnz = 0;
  for (int m = 0; m < M; ++m)
    for (int k = 0; k < K; ++k)
      if (std::fabs(A[(size_t)m * K + k]) > thr) {
        sup[m][k] = 1;
        ++nnz;
      }
  const double density = (double)nnz / ((double)M * K);
  // ---- chunks: a function of the sources' row counts alone.  (A streamed operator may cut a source into lower chunks, `step` rows
  // each, so that a chunk's operator blocks fit a ring stage: steps are multiples of 8 and the k-blocks are formed inside groups of
  // 8 rows, so the sequence of k-blocks -- the summation order -- is the same for every step.)
  std::vector<ChunkDesc> chunks;
  std::vector<int> chunk_k0;   // column of A behind stage row 0 of the chunk
  int src_step[PANEL_MAXSRC] = {0, 0};
  auto make_chunks = [&](int step_cap) {
    chunks.clear();
    chunk_k0.clear();
    int k0 = 0, si = 0;
    for (auto &s : srcs) {
      const int step = std::min(panel_chunk_step(s.rows, std::max(step_cap, PANEL_KCMAX)), step_cap);
      src_step[si] = step;
      for (int r = 0; r < s.rows; r += step) {
        chunks.push_back(ChunkDesc{si, r, std::min(step, s.rows - r), step, 0, 0, 0, 0});
        chunk_k0.push_back(k0 + r);
      }
      k0 += s.rows;
      ++si;
    }
  };
  // Long stacked operands (the fused divergence operator of prisms at p >= 4: K = 330) take chunks of at most 32 rows: their packed image
  // leaves the ring only two 40-row stages per warp group, and a third stage is worth more than the per-chunk overhead it costs
  // (pri S8-S10 FP64 0.82 -> 0.72 ms; every shorter operand is slower with lower chunks; in FP32 the image is half the size and the
  // rule does not apply).  A function of the operator alone.
  make_chunks((f64 && srcs.size() == 2 && K >= 300) ? 32 : PANEL_KCMAX);
  int nchunks = (int)chunks.size();
  if (nchunks > PANEL_MAXCHUNKS) return false;

  // ---- rows -> groups of 8, for a given packing
  auto make_order = [&](bool sparse) {
    std::vector<int> order;   // virtual row -> actual row or -1
    if (opt.triple) {
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
    return order;
  };
  if (opt.triple) FR_REQUIRE(M % 3 == 0, "triple packing needs M divisible by 3");
  // per (group, chunk): the stage rows with a non-zero in the group
  auto make_lists = [&](const std::vector<int> &order) {
    const int G = (int)order.size() / 8;
    std::vector<std::vector<std::vector<int>>> lists(G, std::vector<std::vector<int>>(nchunks));
    for (int g = 0; g < G; ++g)
      for (int c = 0; c < nchunks; ++c)
        for (int kk = 0; kk < chunks[c].nrows; ++kk) {
          bool any = false;
          for (int r = 0; r < 8 && !any; ++r) {
            const int m = order[8 * g + r];
            if (m >= 0 && sup[m][chunk_k0[c] + kk]) any = true;
          }
          if (any) lists[g][c].push_back(kk);
        }
    return lists;
  };
  // ---- packing: k-lists when they save at least 15 % of the multiplies of the dense packing (a function of the operator alone).
  // A streamed operator is always packed densely (its blocks must be one contiguous range per chunk).
  bool sparse = false;
  std::vector<int> order = make_order(false);
  std::vector<std::vector<std::vector<int>>> lists;
  if (opt.allow_sparse && !opt.stream && density < 0.95) {
    std::vector<int> so = make_order(true);
    auto sl = make_lists(so);
    double ds = 0, dd = 0;
    for (auto &g : sl)
      for (auto &l : g) ds += f64 ? (double)((l.size() + 3) / 4) : (double)l.size();
    for (int c = 0; c < nchunks; ++c) dd += (f64 ? (double)dense_blocks_f64(chunks[c].nrows).size() : (double)chunks[c].nrows) * (order.size() / 8);
    if (ds < 0.85 * dd) {
      sparse = true;
      order = so;
      lists = sl;
    }
  }
  // k-list operators take chunks of up to 128 rows (one chunk per operand of configs 1-3).  FP64: a group's k-list is cut into blocks of four
  // per chunk, so every chunk boundary leaves a partly filled block -- fewer chunks, fewer multiplies (pri S3+S4 0.95 -> 0.82 ms, tet S3+S4
  // 1.29 -> 1.26; dense operators are slower with chunks above 40 rows, their block count does not depend on it).  Still a function of the
  // operator alone: if no geometry fits shared memory with the high chunks, all candidates use the default ones.  FP32: see the geometry loop.
  const int default_cap = (f64 && srcs.size() == 2 && K >= 300) ? 32 : PANEL_KCMAX;
  bool high_chunks = f64 && sparse && !opt.stream && default_cap == PANEL_KCMAX;
  if (high_chunks) {
    make_chunks(128);
    nchunks = (int)chunks.size();
    lists = make_lists(order);
  }
  const int G = (int)order.size() / 8;

  // ---- geometry: candidate k = the k-th geometry of the list that fits shared memory
  const std::vector<PanelGeom> geoms = list_geoms<T>(G, opt.min_ne, opt.max_ne, opt.triple, !sparse);
  if (opt.cand < 0) return false;
  int nfit = 0;
  for (int attempt = 0; attempt < 2; ++attempt) {
  if (attempt == 1) {
    if (!high_chunks || nfit > 0) break;   // the candidate does not exist, or there is nothing else to try
    high_chunks = false;
    make_chunks(default_cap);
    nchunks = (int)chunks.size();
    lists = make_lists(order);
  }
  for (const PanelGeom &geo : geoms) {
    size_t smem_total = smem_total_in;
    if (geo.occ == 2) smem_total = smem_total / 2 - 1024;
    const int WR = geo.WR, NIT = geo.NIT, NS = WR * NIT;
    // cost of each group (blocks it executes) and LPT assignment of group units (1 or 3 groups) to row-warps
    std::vector<long long> gcost(G, 0);
    for (int g = 0; g < G; ++g)
      for (int c = 0; c < nchunks; ++c) {
        const int n = sparse ? (int)lists[g][c].size() : chunks[c].nrows;
        gcost[g] += f64 ? (n + 3) / 4 * 4 : n;
      }
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
    std::vector<int> rowmap(NS * 8, -1);
    for (int s = 0; s < NS; ++s)
      if (slot_group[s] >= 0)
        for (int r = 0; r < 8; ++r) {
          const int m = order[8 * slot_group[s] + r];
          rowmap[s * 8 + r] = (m >= 0 && opt.row_ids) ? opt.row_ids[m] : m;
        }
    auto aval = [&](int m, int col) {
      if (m < 0) return 0.0;
      const double v = A[(size_t)m * K + col];
      return std::fabs(v) > thr ? v : 0.0;
    };
    // every array is copied to shared memory by one bulk copy: sizes are multiples of 16 bytes
    auto pad16 = [](auto &v) {
      using E = typename std::remove_reference<decltype(v[0])>::type;
      while ((v.size() * sizeof(E)) % 16) v.push_back(E());
    };
    pad16(rowmap);
    const uint32_t rs32 = (uint32_t)geo.NE * 4u;   // FP32: bytes between stage rows
    const size_t ablk = (size_t)NS * (f64 ? 256 : 32);   // bytes of one packed block row (all slots)
    std::vector<T> vals;
    std::vector<uint32_t> idx;
    std::vector<int> off;
    long long macs = 0;
    int nblk = 0, nstage = 0;
    size_t smem_op = 0, stage_bytes = 0;
    // ---- pack for the current chunks; false if the result does not fit
    auto pack = [&]() {
      vals.clear();
      idx.clear();
      off.assign(sparse ? nchunks * NS + 1 : 1, 0);
      macs = 0;
      nblk = 0;
      if (!sparse) {
        // dense: blocks ordered (chunk, k-block, slot); the rows of a k-block come from the row table idx[block][4] (FP64)
        for (int c = 0; c < nchunks; ++c) {
          chunks[c].base = nblk / NS;
          if (f64) {
            const auto blocks = dense_blocks_f64(chunks[c].nrows);
            chunks[c].nblk = (int)blocks.size();
            for (auto &b : blocks) {
              for (int j = 0; j < 4; ++j) idx.push_back(swz_row_offset(j < (int)b.size() ? b[j] : b[0]));
              for (int s = 0; s < NS; ++s) {
                const int g = slot_group[s];
                for (int lane = 0; lane < 32; ++lane) {
                  const int r = lane >> 2, j = lane & 3;
                  const int m = g >= 0 ? order[8 * g + r] : -1;
                  vals.push_back((T)(j < (int)b.size() ? aval(m, chunk_k0[c] + b[j]) : 0.0));
                }
                if (g >= 0) macs += 32;
                ++nblk;
              }
            }
          } else {
            chunks[c].nblk = chunks[c].nrows;
            for (int k = 0; k < chunks[c].nrows; ++k)
              for (int s = 0; s < NS; ++s) {
                const int g = slot_group[s];
                for (int r = 0; r < 8; ++r) vals.push_back((T)aval(g >= 0 ? order[8 * g + r] : -1, chunk_k0[c] + k));
                if (g >= 0) macs += 8;
                ++nblk;
              }
          }
        }
      } else {
        for (int c = 0; c < nchunks; ++c)
          for (int s = 0; s < NS; ++s) {
            off[c * NS + s] = nblk;
            const int g = slot_group[s];
            if (g < 0) continue;
            const std::vector<int> &L = lists[g][c];
            if (f64) {
              for (auto &b : sparse_blocks_f64(L)) {
                for (int j = 0; j < 4; ++j) idx.push_back(swz_row_offset(j < (int)b.size() ? b[j] : b[0]));
                for (int lane = 0; lane < 32; ++lane) {
                  const int r = lane >> 2, j = lane & 3;
                  vals.push_back((T)(j < (int)b.size() ? aval(order[8 * g + r], chunk_k0[c] + b[j]) : 0.0));
                }
                ++nblk;
                macs += 32;
              }
            } else {
              for (int kk : L) {
                idx.push_back((uint32_t)kk * rs32);
                for (int r = 0; r < 8; ++r) vals.push_back((T)aval(order[8 * g + r], chunk_k0[c] + kk));
                ++nblk;
                macs += 8;
              }
            }
          }
        off[nchunks * NS] = nblk;
      }
      // the sparse multiply loop prefetches two blocks ahead: two all-zero blocks close the arrays (not counted in nblk)
      for (int d = 0; d < 2; ++d) {
        for (int j = 0; j < (f64 ? 4 : 1); ++j) idx.push_back(0u);
        for (int j = 0; j < (f64 ? 32 : 8); ++j) vals.push_back(T(0));
      }
      pad16(vals);
      pad16(idx);
      pad16(off);
      smem_op = (opt.stream ? 0 : vals.size() * sizeof(T)) + idx.size() * 4 + off.size() * 4 + rowmap.size() * 4 + chunks.size() * sizeof(ChunkDesc);
      if (smem_op > smem_budget) return false;
      size_t bmax = 0, amax_b = 0;
      for (auto &c : chunks) {
        bmax = std::max(bmax, (size_t)PV * geo.NE * c.step * sizeof(T));
        amax_b = std::max(amax_b, (size_t)c.nblk * ablk);
      }
      const size_t a_off = (bmax + 127) / 128 * 128;   // = PanelOp::a_off(): one source, so bmax is the box of src_step[0] rows
      stage_bytes = (a_off + (opt.stream ? amax_b : 0) + 1023) / 1024 * 1024;
      // 1 kB to align the ring, the ring, 256 B of mbarriers
      const size_t fixed = 1024 + (smem_op + 1023) / 1024 * 1024 + 256;
      if (fixed + 2 * geo.NG * stage_bytes > smem_total) return false;
      nstage = std::min((int)((smem_total - fixed) / (geo.NG * stage_bytes)), PANEL_MAXSTAGE);
      return true;
    };
    bool fits = false;
    if (!f64 && sparse && !opt.stream) {
      // FP32 k-lists hold single rows, in increasing order whatever the chunking: the chunk height may follow the geometry without
      // changing a bit of the result.  The highest chunks (fewest chunk boundaries: pri S3+S4 0.59 -> 0.53 ms) that leave this
      // geometry's panel width a ring of two stages.
      for (int cap : {128, 96, 64, PANEL_KCMAX}) {
        make_chunks(cap);
        nchunks = (int)chunks.size();
        lists = make_lists(order);
        fits = pack();
        if (fits) break;
      }
    } else if (!opt.stream) {
      fits = pack();
    } else {
      // the highest chunks that leave a ring of four stages; failing that, the deepest ring any chunk height gives
      int best_step = 0, best_stages = 0;
      for (int step = PANEL_KCMAX; step >= 8; step -= 8) {
        make_chunks(step);
        nchunks = (int)chunks.size();
        if (nchunks > PANEL_MAXCHUNKS || !pack()) continue;
        if (nstage > best_stages) {
          best_stages = nstage;
          best_step = step;
        }
        if (nstage >= 4) break;
      }
      if (best_step) {
        make_chunks(best_step);
        nchunks = (int)chunks.size();
        fits = pack();
      }
    }
    if (!fits) continue;
    if (nfit++ != opt.cand) continue;
    if (getenv("FRB_NSTAGE")) nstage = std::max(2, std::min(nstage, atoi(getenv("FRB_NSTAGE"))));
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
    p.nchunks = nchunks;
    p.NS = NS;
    p.nstage = nstage;
    p.stage_bytes = (int)stage_bytes;
    p.nblk = nblk;
    p.nidx = (int)idx.size();
    p.nsrc = (int)srcs.size();
    for (int i = 0; i < p.nsrc; ++i) {
      p.src_rows[i] = srcs[i].rows;
      p.src_step[i] = src_step[i];
    }
#ifdef FRB_DEBUG_KNOBS
    p.dbg = getenv("FRB_PANEL_DBG") ? atoi(getenv("FRB_PANEL_DBG")) : 0;
    if (getenv("FRB_PANEL_VERBOSE"))
      fprintf(stderr, "panel_op %s M=%d K=%d %s%s G=%d WR=%d WC=%d NIT=%d CX=%d NE=%d NG=%d occ=%d warps=%d+%d nchunks=%d nblk=%d smem_op=%zu stage=%zu x %d density=%.2f macs/col=%.0f (dense %d)\n",
              f64 ? "f64" : "f32", M, K, sparse ? "sparse" : "dense", opt.stream ? " streamed" : "", G, WR, geo.WC, NIT, geo.CX, geo.NE, geo.NG, geo.occ,
              geo.NG * WR * geo.WC, geo.NG, nchunks, nblk, smem_op, stage_bytes, nstage, density, (double)macs, M * K);
#endif
    p.sparse = sparse ? 1 : 0;
    p.macs_per_col = (double)macs;
    p.density = density;
    p.smem_op = smem_op;
    p.bytes_vals = opt.stream ? 0 : vals.size() * sizeof(T);
    p.bytes_idx = idx.size() * 4;
    p.bytes_off = off.size() * 4;
    p.bytes_rowmap = rowmap.size() * 4;
    p.bytes_chunks = chunks.size() * sizeof(ChunkDesc);
    auto up = [](auto *&dst, const auto &h) {
      using E = typename std::remove_reference<decltype(h[0])>::type;
      FR_CUDA_TRY(cudaMalloc((void **)&dst, h.size() * sizeof(E)));
      FR_CUDA_TRY(cudaMemcpy((void *)dst, h.data(), h.size() * sizeof(E), cudaMemcpyHostToDevice));
    };
    up(p.vals, vals);
    up(p.idx, idx);
    up(p.off, off);
    up(p.rowmap, rowmap);
    up(p.chunks, chunks);
    return true;
  }
  }
  return false;
}

template <typename T>
inline size_t panel_smem_bytes(const PanelOp<T> &op) {
  return 1024 + (op.smem_op + 1023) / 1024 * 1024 + (size_t)op.NG * op.nstage * op.stage_bytes + 256;
}

// ------------------------------------------------------------------------------------------------ device side
#ifdef __CUDACC__

__device__ __forceinline__ void prefetch_l2(const void *p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }

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
__device__ __forceinline__ void op_smem_carve(char *base, const PanelOp<T> &op, OpSmem<T> &v) {
  v.vals = reinterpret_cast<const T *>(base);
  base += op.bytes_vals;
  v.idx = reinterpret_cast<const uint32_t *>(base);
  base += op.bytes_idx;
  v.off = reinterpret_cast<const int *>(base);
  base += op.bytes_off;
  v.rowmap = reinterpret_cast<const int *>(base);
  base += op.bytes_rowmap;
  v.chunks = reinterpret_cast<const ChunkDesc *>(base);
}

// ---- accumulators and the multiply-accumulate core.  A stage holds the chunk as planes (tma.cuh):
//   FP64: plane(v, cb16) = v*(NE/16) + cb16, `pp` = step*128 bytes each, rows of 16 doubles, 128-byte swizzle;
//   FP32: plane(v) of step rows of NE floats.
// PACKED selects the FP32 form (packed pairs / scalar); FP64 has one form
template <typename T, int NIT, int CX, bool PACKED = true>
struct Acc;

// FP64: per slot, CX column blocks of 8 elements x 5 variables, one m8n8k4 C fragment (2 doubles) each.
template <int NIT, int CX, bool PACKED>
struct Acc<double, NIT, CX, PACKED> {
  double c[NIT][CX][PV][2];
  __device__ __forceinline__ void zero() {
#pragma unroll
    for (int i = 0; i < NIT; ++i)
#pragma unroll
      for (int b = 0; b < CX; ++b)
#pragma unroll
        for (int v = 0; v < PV; ++v) c[i][b][v][0] = c[i][b][v][1] = 0.0;
  }
  // Per-lane constants of the B-fragment loads: lane = (column c = lane/4 of the 8-column block, k = lane%4).  Column block
  // cbi = wc*CX + cb of the panel sits in 16-block cbi/2, half cbi%2: byte (half*4 + c/2)*16 + (c%2)*8 of the 128-byte line,
  // XORed with the line's swizzle term, which the row offsets of idx carry in bits 4..6.
  __device__ __forceinline__ static uint32_t lane_term(int cbi, int lane) {
    const int c = lane >> 2;
    return ((uint32_t)(((cbi & 1) << 2) | (c >> 1)) << 4) | ((uint32_t)(c & 1) << 3);
  }
  // Sparse operator: the warp's blocks of this chunk are contiguous across its NIT slots, so one software pipeline runs
  // through all of them: operator value and row offset are fetched two blocks ahead, the B fragments one block ahead of the
  // DMMAs that consume them.
  __device__ __forceinline__ void mac_chunk(const OpSmem<double> &A, int chunk, const ChunkDesc &cd, int NS, int slot0, const char *stage,
                                            int NE, int wc, int lane) {
    const uint32_t pp = (uint32_t)cd.step * 128u;
    const uint32_t vs = (uint32_t)(NE >> 4) * pp;
    uint32_t lt[CX];
    const char *pl[CX];
#pragma unroll
    for (int cb = 0; cb < CX; ++cb) {
      const int cbi = wc * CX + cb;
      lt[cb] = lane_term(cbi, lane);
      pl[cb] = stage + (uint32_t)(cbi >> 1) * pp;
    }
    const char *av = reinterpret_cast<const char *>(A.vals) + lane * 8;
    const char *ai = reinterpret_cast<const char *>(A.idx) + (lane & 3) * 4;
    const int *offp = A.off + chunk * NS + slot0;
    int b = offp[0];
    double a0 = *reinterpret_cast<const double *>(av + (uint32_t)b * 256u);
    double a1 = *reinterpret_cast<const double *>(av + (uint32_t)b * 256u + 256u);
    uint32_t ro1 = *reinterpret_cast<const uint32_t *>(ai + (uint32_t)b * 16u + 16u);
    double bf0[PV][CX];
    {
      const uint32_t ro0 = *reinterpret_cast<const uint32_t *>(ai + (uint32_t)b * 16u);
#pragma unroll
      for (int cb = 0; cb < CX; ++cb) {
        const char *bp = pl[cb] + (ro0 ^ lt[cb]);
#pragma unroll
        for (int v = 0; v < PV; ++v) bf0[v][cb] = *reinterpret_cast<const double *>(bp + v * vs);
      }
    }
#pragma unroll
    for (int i = 0; i < NIT; ++i) {
      const int bend = offp[i + 1];
#pragma unroll 2
      for (; b < bend; ++b) {
        double bf1[PV][CX];
#pragma unroll
        for (int cb = 0; cb < CX; ++cb) {
          const char *bp = pl[cb] + (ro1 ^ lt[cb]);
#pragma unroll
          for (int v = 0; v < PV; ++v) bf1[v][cb] = *reinterpret_cast<const double *>(bp + v * vs);
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
  // Dense operator: the NIT row groups of the warp share the chunk's k-blocks, so the B fragments of a k-block are loaded
  // once and feed NIT x 5 x CX DMMAs; the block's four stage rows come from the row table.
  // STREAM: the chunk's packed blocks sit behind the chunk in the stage (offset a_off) instead of in the resident image.
  template <bool STREAM>
  __device__ __forceinline__ void mac_dense(const OpSmem<double> &A, const ChunkDesc &cd, int NS, int slot0, const char *stage, int NE,
                                            int wc, int lane, int a_off) {
    const uint32_t pp = (uint32_t)cd.step * 128u;
    const uint32_t vs = (uint32_t)(NE >> 4) * pp;
    uint32_t lt[CX];
    const char *pl[CX];
#pragma unroll
    for (int cb = 0; cb < CX; ++cb) {
      const int cbi = wc * CX + cb;
      lt[cb] = lane_term(cbi, lane);
      pl[cb] = stage + (uint32_t)(cbi >> 1) * pp;
    }
    const char *av = STREAM ? stage + a_off + ((uint32_t)slot0 * 32u + lane) * 8u
                            : reinterpret_cast<const char *>(A.vals) + ((uint32_t)(cd.base * NS + slot0) * 32u + lane) * 8u;
    const uint32_t *rt = A.idx + cd.base * 4 + (lane & 3);
    const uint32_t as = (uint32_t)NS * 256u;
    const int nb = cd.nblk;
#pragma unroll 2
    for (int b = 0; b < nb; ++b) {
      const uint32_t ro = rt[b * 4];
      double bf[PV][CX];
#pragma unroll
      for (int cb = 0; cb < CX; ++cb) {
        const char *bp = pl[cb] + (ro ^ lt[cb]);
#pragma unroll
        for (int v = 0; v < PV; ++v) bf[v][cb] = *reinterpret_cast<const double *>(bp + v * vs);
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
  static constexpr int EW = 2;   // consecutive elements per foreach_tile call
  static constexpr int ROWS = 1; // rows per thread per slot
  static constexpr int NSLOT = NIT;
};

// ---- packed FP32 pairs: fma.rn.f32x2 (FFMA2, sm_100) does two IEEE FP32 fused multiply-adds per instruction -- the same
// results as two FFMA at the same pipe rate for half the issue slots, which is what the FP32 multiply loops are short of.
__device__ __forceinline__ void ffma2(unsigned long long &c, unsigned long long a, unsigned long long b) {
  asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(c) : "l"(a), "l"(b));
}
__device__ __forceinline__ unsigned long long pack2(float lo, float hi) {
  unsigned long long r;
  asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
  return r;
}
__device__ __forceinline__ void unpack2(unsigned long long v, float &lo, float &hi) {
  asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}

// FP32: per slot, 8 rows x 5 variables x CX elements per lane; rows 2q and 2q+1 share a register pair (the operator's packed
// columns hold them next to each other, so a pair of operator values is one 64-bit half of the LDS.128 that fetches it).
template <int NIT, int CX>
struct Acc<float, NIT, CX, true> {
  unsigned long long c[NIT][4][PV][CX];
  __device__ __forceinline__ void zero() {
#pragma unroll
    for (int i = 0; i < NIT; ++i)
#pragma unroll
      for (int q = 0; q < 4; ++q)
#pragma unroll
        for (int v = 0; v < PV; ++v)
#pragma unroll
          for (int j = 0; j < CX; ++j) c[i][q][v][j] = 0ull;
  }
  // the chunk's B values of one stage row for this lane, each duplicated into both halves of a pair
  __device__ __forceinline__ static void load_b(const char *bp, uint32_t vs, unsigned long long (&bd)[PV][CX]) {
#pragma unroll
    for (int v = 0; v < PV; ++v) {
      if (CX == 2) {
        const float2 t = *reinterpret_cast<const float2 *>(bp);
        bd[v][0] = pack2(t.x, t.x);
        bd[v][CX - 1] = pack2(t.y, t.y);
      } else {
        const float t = *reinterpret_cast<const float *>(bp);
        bd[v][0] = pack2(t, t);
      }
      bp += vs;
    }
  }
  // 8 operator values (one packed column of a slot) times the row of B
  __device__ __forceinline__ void mac_col(int i, const char *ap, const unsigned long long (&bd)[PV][CX]) {
    const ulonglong2 a01 = *reinterpret_cast<const ulonglong2 *>(ap);
    const ulonglong2 a23 = *reinterpret_cast<const ulonglong2 *>(ap + 16);
    const unsigned long long aq[4] = {a01.x, a01.y, a23.x, a23.y};
#pragma unroll
    for (int q = 0; q < 4; ++q)
#pragma unroll
      for (int v = 0; v < PV; ++v)
#pragma unroll
        for (int j = 0; j < CX; ++j) ffma2(c[i][q][v][j], aq[q], bd[v][j]);
  }
  __device__ __forceinline__ void mac_chunk(const OpSmem<float> &A, int chunk, const ChunkDesc &cd, int NS, int slot0, const char *stage,
                                            int NE, int wc, int lane) {
    const char *bcol = stage + (uint32_t)(wc * 32 * CX + lane * CX) * 4u;
    const char *avp = reinterpret_cast<const char *>(A.vals);
    const uint32_t vs = (uint32_t)cd.step * (uint32_t)NE * 4u;
#pragma unroll
    for (int i = 0; i < NIT; ++i) {
      const int b0 = A.off[chunk * NS + slot0 + i], b1 = A.off[chunk * NS + slot0 + i + 1];
#pragma unroll 2
      for (int b = b0; b < b1; ++b) {
        unsigned long long bd[PV][CX];
        load_b(bcol + A.idx[b], vs, bd);
        mac_col(i, avp + (uint32_t)b * 32u, bd);
      }
    }
  }
  // Dense operator: one B row feeds the NIT row groups of the warp.
  template <bool STREAM>
  __device__ __forceinline__ void mac_dense(const OpSmem<float> &A, const ChunkDesc &cd, int NS, int slot0, const char *stage, int NE,
                                            int wc, int lane, int a_off) {
    const char *bp0 = stage + (uint32_t)(wc * 32 * CX + lane * CX) * 4u;
    const char *ap0 = STREAM ? stage + a_off + (uint32_t)slot0 * 32u
                             : reinterpret_cast<const char *>(A.vals) + (uint32_t)(cd.base * NS + slot0) * 32u;
    const uint32_t rs = (uint32_t)NE * 4u, vs = (uint32_t)cd.step * rs, as = (uint32_t)NS * 32u;
#pragma unroll 2
    for (int k = 0; k < cd.nrows; ++k) {
      unsigned long long bd[PV][CX];
      load_b(bp0 + (uint32_t)k * rs, vs, bd);
      const char *ap = ap0 + (uint32_t)k * as;
#pragma unroll
      for (int i = 0; i < NIT; ++i) mac_col(i, ap + i * 32, bd);
    }
  }
  // rows 2q and 2q+1 of slot i as float tiles
  __device__ __forceinline__ void rows_of(int i, int q, float (&t0)[PV][CX], float (&t1)[PV][CX]) const {
#pragma unroll
    for (int v = 0; v < PV; ++v)
#pragma unroll
      for (int j = 0; j < CX; ++j) unpack2(c[i][q][v][j], t0[v][j], t1[v][j]);
  }
  template <typename F>
  __device__ __forceinline__ void foreach_tile(int wc, int lane, F &&f) {
#pragma unroll
    for (int i = 0; i < NIT; ++i)
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        float t0[PV][CX], t1[PV][CX];
        rows_of(i, q, t0, t1);
        f(i, 2 * q, wc * 32 * CX + lane * CX, t0);
        f(i, 2 * q + 1, wc * 32 * CX + lane * CX, t1);
      }
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
      for (int q = 0; q < 4; ++q) {
        float a0[PV][CX], a1[PV][CX], b0[PV][CX], b1[PV][CX], c0[PV][CX], c1[PV][CX];
        rows_of(3 * t, q, a0, a1);
        rows_of(3 * t + 1, q, b0, b1);
        rows_of(3 * t + 2, q, c0, c1);
        f(t, 2 * q, wc * 32 * CX + lane * CX, a0, b0, c0);
        f(t, 2 * q + 1, wc * 32 * CX + lane * CX, a1, b1, c1);
      }
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

// FP32, scalar form (FFMA): per slot, 8 rows x 5 variables x CX elements per lane.  Kept for the gradient kernels, whose 12-warp /
// 168-register budget has no room for the register-pair alignment of the packed form (it spills into the multiply loop there).
template <int NIT, int CX>
struct Acc<float, NIT, CX, false> {
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
  __device__ __forceinline__ void mac_chunk(const OpSmem<float> &A, int chunk, const ChunkDesc &cd, int NS, int slot0, const char *stage,
                                            int NE, int wc, int lane) {
    const char *bcol = stage + (uint32_t)(wc * 32 * CX + lane * CX) * 4u;
    const char *avp = reinterpret_cast<const char *>(A.vals);
    const uint32_t vs = (uint32_t)cd.step * (uint32_t)NE * 4u;
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
  template <bool STREAM>
  __device__ __forceinline__ void mac_dense(const OpSmem<float> &A, const ChunkDesc &cd, int NS, int slot0, const char *stage, int NE,
                                            int wc, int lane, int a_off) {
    const char *bp0 = stage + (uint32_t)(wc * 32 * CX + lane * CX) * 4u;
    const char *ap0 = STREAM ? stage + a_off + (uint32_t)slot0 * 32u
                             : reinterpret_cast<const char *>(A.vals) + (uint32_t)(cd.base * NS + slot0) * 32u;
    const uint32_t rs = (uint32_t)NE * 4u, vs = (uint32_t)cd.step * rs, as = (uint32_t)NS * 32u;
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
