// Operator product C <- c1*A*B + c2*C (eq. 1): A = small constant operator (M x K),
// B (K x N) and C (M x N) wide row-major state matrices -- the block-by-panel (GEBP) case of PAPER.md:39.
//
// B200 design (not the paper's: it defers to cuBLAS): every column of B is independent, so a
// persistent CTA owns column panels (the decomposition the paper's OpenMP backend found best).
//   * the operator slab (transposed, zero padded, [K][TY*MT]) stays resident in shared memory for the whole
//     kernel when it fits, so L2->SM traffic is the B panel only;
//   * B panels stream global->shared through a 4-stage cp.async ring that runs across panel boundaries
//     (16-byte, fully coalesced row segments; K and N tails zero-filled by the copy itself);
//   * each thread keeps an MT x CT register tile (CT = one 16-byte vector of columns), A is read as warp-wide
//     broadcast vectors, B as conflict-free vectors; FP64 uses DFMA, FP32 FFMA (no TF32: the 2e-5 parity bound
//     and reading R15 exclude it; tcgen05 has no FP64 kind);
//   * C is written once with 16-byte coalesced stores; c2 != 0 reads it once.
#include <algorithm>
#include <mutex>

#include "common.cuh"
#include "panel.cuh"

namespace frb {

template <typename T>
bool panel_gemm_build(PanelOp<T> &op, int M, int K, const double *A, int cand = 0, double drop_rel = 1.4210854715202004e-14, int stream = 0);
template <typename T>
void panel_gemm_run(const PanelOp<T> &op, long long N, T c1, const T *B, long long ldb, long long bsB, T c2, T *C,
                    long long ldc, long long bsC, int nbatch, cudaStream_t s);

namespace {

constexpr int KC = 16;      // K rows per pipeline stage
constexpr int NSTAGE = 4;   // cp.async ring depth

template <typename T>
struct VecT;
template <>
struct VecT<double> {
  using type = double2;
  static constexpr int CT = 2;
};
template <>
struct VecT<float> {
  using type = float4;
  static constexpr int CT = 4;
};

template <typename T>
struct GemmArgs {
  int M, K, nchunks, nrb, nbatch;
  long long N, ntn;            // columns, column tiles per batch
  const T *At;                 // [nrb][Kpad][MTILE]
  const T *B;
  T *C;
  long long ldb, ldc, bsB, bsC;
  T c1, c2;
};

__device__ __forceinline__ void cp_async16(void *smem, const void *gmem, int src_bytes) {
  unsigned s = (unsigned)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(s), "l"(gmem), "r"(src_bytes));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::); }
template <int N>
__device__ __forceinline__ void cp_async_wait() {
  asm volatile("cp.async.wait_group %0;\n" ::"n"(N));
}

template <typename T, int MT, int TY, bool RESIDENT>
__global__ void __launch_bounds__(32 * TY) k_gemm(const __grid_constant__ GemmArgs<T> a) {
  using V = typename VecT<T>::type;
  constexpr int CT = VecT<T>::CT;
  constexpr int NT = 32 * CT;
  constexpr int MTILE = TY * MT;
  constexpr int NTHREADS = 32 * TY;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  T *Bs = reinterpret_cast<T *>(smem_raw);                         // [NSTAGE][KC][NT]
  T *As = Bs + NSTAGE * KC * NT;                                   // resident: [Kpad][MTILE]; else [NSTAGE][KC][MTILE]

  const int tx = threadIdx.x, ty = threadIdx.y;
  const int tid = ty * 32 + tx;
  const int rb = blockIdx.x % a.nrb;
  const long long lane = blockIdx.x / a.nrb;
  const long long stride = gridDim.x / a.nrb;
  const long long ntiles = a.ntn * a.nbatch;
  const long long mytiles = lane < ntiles ? (ntiles - lane + stride - 1) / stride : 0;
  const long long total = mytiles * a.nchunks;
  const int Kpad = a.nchunks * KC;
  const T *At = a.At + (long long)rb * Kpad * MTILE;

  if (RESIDENT) {
    const int npieces = Kpad * MTILE * (int)sizeof(T) / 16;
    for (int p = tid; p < npieces; p += NTHREADS)
      cp_async16(reinterpret_cast<char *>(As) + 16 * p, reinterpret_cast<const char *>(At) + 16 * p, 16);
  }

  auto issue = [&](long long q) {
    const long long tile = lane + (q / a.nchunks) * stride;
    const int c = (int)(q % a.nchunks);
    const int st = (int)(q % NSTAGE);
    const long long batch = tile / a.ntn;
    const long long col0 = (tile % a.ntn) * NT;
    const T *Bb = a.B + batch * a.bsB;
    T *bs = Bs + st * KC * NT;
#pragma unroll
    for (int p = tid; p < KC * 32; p += NTHREADS) {
      const int row = p >> 5, pc = p & 31;
      const int k = c * KC + row;
      const long long col = col0 + pc * CT;
      long long rem = (a.N - col) * (long long)sizeof(T);
      int nb = (k < a.K) ? (rem >= 16 ? 16 : (rem > 0 ? (int)rem : 0)) : 0;
      const T *src = nb > 0 ? Bb + (long long)k * a.ldb + col : a.B;
      cp_async16(bs + row * NT + pc * CT, src, nb);
    }
    if (!RESIDENT) {
      T *as = As + st * KC * MTILE;
      constexpr int PPR = MTILE * (int)sizeof(T) / 16;             // 16-byte pieces per row
      for (int p = tid; p < KC * PPR; p += NTHREADS) {
        const int row = p / PPR, pc = p % PPR;
        cp_async16(reinterpret_cast<char *>(as + row * MTILE) + 16 * pc,
                   reinterpret_cast<const char *>(At + (long long)(c * KC + row) * MTILE) + 16 * pc, 16);
      }
    }
  };

  for (int q = 0; q < NSTAGE - 1; ++q) {
    if (q < total) issue(q);
    cp_async_commit();
  }

  T acc[MT][CT];
#pragma unroll
  for (int i = 0; i < MT; ++i)
#pragma unroll
    for (int j = 0; j < CT; ++j) acc[i][j] = T(0);

  for (long long q = 0; q < total; ++q) {
    cp_async_wait<NSTAGE - 2>();
    __syncthreads();
    if (q + NSTAGE - 1 < total) issue(q + NSTAGE - 1);
    cp_async_commit();

    const int c = (int)(q % a.nchunks);
    const int st = (int)(q % NSTAGE);
    const T *bs = Bs + st * KC * NT + tx * CT;
    const T *as = (RESIDENT ? As + c * KC * MTILE : As + st * KC * MTILE) + ty * MT;
    const int kend = min(KC, a.K - c * KC);
#pragma unroll 4
    for (int kk = 0; kk < kend; ++kk) {
      T bv[CT];
      *reinterpret_cast<V *>(bv) = *reinterpret_cast<const V *>(bs + kk * NT);
      T av[MT];
      // warp-wide broadcast reads of the operator column; vector width limited by the alignment of ty*MT
      constexpr int AV = (MT % CT == 0) ? CT : 2;
      static_assert(MT % 2 == 0, "MT must be even");
#pragma unroll
      for (int i = 0; i < MT; i += AV) {
        if (AV == CT) {
          *reinterpret_cast<V *>(av + i) = *reinterpret_cast<const V *>(as + kk * MTILE + i);
        } else {
          *reinterpret_cast<float2 *>(av + i) = *reinterpret_cast<const float2 *>(as + kk * MTILE + i);
        }
      }
#pragma unroll
      for (int i = 0; i < MT; ++i)
#pragma unroll
        for (int j = 0; j < CT; ++j) acc[i][j] = fma(av[i], bv[j], acc[i][j]);
    }

    if (c == a.nchunks - 1) {
      const long long tile = lane + (q / a.nchunks) * stride;
      const long long batch = tile / a.ntn;
      const long long col = (tile % a.ntn) * NT + tx * CT;
      T *Cb = a.C + batch * a.bsC;
      const bool full = col + CT <= a.N;
#pragma unroll
      for (int i = 0; i < MT; ++i) {
        const int m = rb * MTILE + ty * MT + i;
        if (m < a.M) {
          T *cp = Cb + (long long)m * a.ldc + col;
          if (full) {
            T out[CT];
            if (a.c2 != T(0)) {
              T old[CT];
              *reinterpret_cast<V *>(old) = *reinterpret_cast<const V *>(cp);
#pragma unroll
              for (int j = 0; j < CT; ++j) out[j] = fma(a.c1, acc[i][j], a.c2 * old[j]);
            } else {
#pragma unroll
              for (int j = 0; j < CT; ++j) out[j] = a.c1 * acc[i][j];
            }
            *reinterpret_cast<V *>(cp) = *reinterpret_cast<V *>(out);
          } else {
#pragma unroll
            for (int j = 0; j < CT; ++j)
              if (col + j < a.N) cp[j] = (a.c2 != T(0)) ? fma(a.c1, acc[i][j], a.c2 * cp[j]) : a.c1 * acc[i][j];
          }
        }
#pragma unroll
        for (int j = 0; j < CT; ++j) acc[i][j] = T(0);
      }
    }
  }
  cp_async_wait<0>();
}

// Grid: persistent CTAs, (resident CTAs per SM from the occupancy calculator) x (SM count), a multiple of the
// number of row blocks, never more than there are panels.
template <typename K, typename T>
void launch_kernel(K k, const GemmPlan<T> &p, const GemmArgs<T> &a, int nthreads, cudaStream_t s) {
  FR_CUDA_TRY(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)p.smem));
  int occ = 1;
  FR_CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k, nthreads, p.smem));
  occ = std::max(1, std::min(occ, 4));
  const long long ntiles = a.ntn * a.nbatch;
  long long lanes = std::max(1, device_sm_count() * occ / p.nrb);
  lanes = std::min(lanes, ntiles);
  k<<<(unsigned)(lanes * p.nrb), dim3(32, nthreads / 32), p.smem, s>>>(a);
  FR_CUDA_TRY(cudaGetLastError());
}

template <typename T, int MT, int TY>
void launch_variant(const GemmPlan<T> &p, const GemmArgs<T> &a, int, cudaStream_t s) {
  if (p.resident) launch_kernel(k_gemm<T, MT, TY, true>, p, a, 32 * TY, s);
  else launch_kernel(k_gemm<T, MT, TY, false>, p, a, 32 * TY, s);
}

template <typename T, int TY>
void launch_ty(const GemmPlan<T> &p, const GemmArgs<T> &a, int grid, cudaStream_t s) {
  switch (p.MT) {
    case 2: launch_variant<T, 2, TY>(p, a, grid, s); break;
    case 4: launch_variant<T, 4, TY>(p, a, grid, s); break;
    case 6: launch_variant<T, 6, TY>(p, a, grid, s); break;
    case 8: launch_variant<T, 8, TY>(p, a, grid, s); break;
    case 10: launch_variant<T, 10, TY>(p, a, grid, s); break;
    case 12: launch_variant<T, 12, TY>(p, a, grid, s); break;
    case 14: launch_variant<T, 14, TY>(p, a, grid, s); break;
    case 16: launch_variant<T, 16, TY>(p, a, grid, s); break;
    default: throw Error{FR_EINVAL, "gemm: bad MT"};
  }
}

}  // namespace

int device_sm_count() {
  // per device: a process may drive several (one context per host thread, include/frb200.h)
  int dev = 0, n = 0;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev);
  return n > 0 ? n : 148;
}

// The panel-kernel forms of a plan.  stream = 0: the operator image stays in shared memory, as row blocks of A (one launch each,
// every block re-reads B) when the whole image does not fit; stream = 1: the operator's packed blocks travel through the TMA ring with
// the chunks of B (panel.cuh), which takes all rows a CTA's accumulators can hold in one pass -- row blocks only beyond that.  The
// fewest blocks that work, rows per block a multiple of 8 and as even as possible.  Both forms give bit-identical results.
template <typename T>
bool plan_variant(GemmPlan<T> &p, int M, int K, const double *A_host, double drop_rel, int stream, int min_parts) {
  for (int np = std::max(1, min_parts); np <= GemmPlan<T>::kMaxParts; ++np) {
    const int per = np == 1 ? M : ((M + np - 1) / np + 7) / 8 * 8;
    if (np > 1 && (long long)per * (np - 1) >= M) continue;
    bool ok = true;
    int n = 0;
    PanelOp<T> *ops[GemmPlan<T>::kMaxParts] = {};
    for (int r0 = 0; r0 < M && ok; r0 += per, ++n) {
      ops[n] = new PanelOp<T>();
      try {
        ok = panel_gemm_build(*ops[n], std::min(per, M - r0), K, A_host + (size_t)r0 * K, 0, drop_rel, stream);
      } catch (...) {
        ok = false;
      }
    }
    if (ok) {
      p.M = M;
      p.K = K;
      if (np == 1) {
        p.pop = ops[0];
      } else {
        p.nparts = n;
        for (int i = 0; i < n; ++i) {
          p.part[i] = ops[i];
          p.part_row0[i] = i * per;
        }
      }
      return true;
    }
    for (int i = 0; i < n; ++i) {
      panel_op_free(*ops[i]);
      delete ops[i];
    }
    if (np == 1 && getenv("FRB_NO_ROWSPLIT")) break;
  }
  return false;
}

template <typename T>
void gemm_plan_build(GemmPlan<T> &p, int M, int K, const double *A_host, double drop_rel) {
  FR_REQUIRE(M > 0 && K > 0 && A_host, "gemm: M, K must be positive and A non-NULL");
  constexpr int CT = VecT<T>::CT;
  p.M = M;
  p.K = K;
  const int force_split = getenv("FRB_FORCE_SPLIT") ? atoi(getenv("FRB_FORCE_SPLIT")) : 0;
  // FRB_GEMM_STREAM: 0 never stream the operator, 1 stream whenever the resident image does not fit; default: the static rule below
  const int stream_mode = getenv("FRB_GEMM_STREAM") ? atoi(getenv("FRB_GEMM_STREAM")) : -1;
  const int min_parts = (force_split >= 2 && M >= 16) ? force_split : 1;
  // preferred: operator resident in shared memory, all rows in one CTA (panel.cuh)
  GemmPlan<T> res, str;
  const bool have_res = plan_variant(res, M, K, A_host, drop_rel, 0, min_parts);
  if (have_res && res.pop) {
    p = res;
    return;
  }
  const bool have_str = stream_mode != 0 && plan_variant(str, M, K, A_host, drop_rel, 1, min_parts);
  if (have_res || have_str) {
    // without timing (fr_gemm; fr_gemm_plan_create times both forms): streamed when the passes over B it saves outweigh twice the
    // rows of C -- the rule that picks the faster form for every operator of BASELINE.json configs[3] (profiles/r02_e_gemm_sweep.md)
    const long long nr = have_res ? res.nparts : 1 << 20, ns = have_str ? std::max(1, str.nparts) : 1 << 20;
    const bool take_str = have_str && (!have_res || stream_mode == 1 || (nr - ns) * K > 2ll * M);
    p = take_str ? str : res;
    if (have_res && take_str) gemm_plan_free(res);
    if (have_str && !take_str) gemm_plan_free(str);
    return;
  }
  double best = 1e300;
  const int tys[3] = {4, 6, 8};
  for (int t = 0; t < 3; ++t)
    for (int mt = 2; mt <= 16; mt += 2) {
      const int tile = tys[t] * mt;
      const int nrb = (M + tile - 1) / tile;
      double score = (double)nrb * tile * (1.0 + 0.15 * (nrb - 1)) - 1e-3 * tys[t];
      if (score < best) {
        best = score;
        p.TY = tys[t];
        p.MT = mt;
        p.nrb = nrb;
      }
    }
  const int MTILE = p.TY * p.MT;
  const int nchunks = (K + KC - 1) / KC;
  const int Kpad = nchunks * KC;
  const size_t bs_bytes = (size_t)NSTAGE * KC * 32 * CT * sizeof(T);
  const size_t slab = (size_t)Kpad * MTILE * sizeof(T);
  p.resident = slab <= 96 * 1024;
  p.smem = bs_bytes + (p.resident ? slab : (size_t)NSTAGE * KC * MTILE * sizeof(T));
  p.ctas_per_sm = (int)std::max<size_t>(1, std::min<size_t>(3, (200 * 1024) / p.smem));
  // register file: 32*TY threads at <= 128 registers
  p.ctas_per_sm = std::min(p.ctas_per_sm, std::max(1, 512 / (32 * p.TY)));
  std::vector<T> At((size_t)p.nrb * Kpad * MTILE, T(0));
  for (int m = 0; m < M; ++m) {
    const int rb = m / MTILE, mm = m % MTILE;
    for (int k = 0; k < K; ++k) {
      const double v = A_host[(size_t)m * K + k];
      FR_REQUIRE(v == v && v - v == 0.0, "gemm: operator contains non-finite entries");
      At[((size_t)rb * Kpad + k) * MTILE + mm] = (T)v;
    }
  }
  FR_CUDA_TRY(cudaMalloc(&p.At, At.size() * sizeof(T)));
  FR_CUDA_TRY(cudaMemcpy(p.At, At.data(), At.size() * sizeof(T), cudaMemcpyHostToDevice));
}

// Time the launch geometries of a plan's panel operator on scratch matrices larger than L2 and keep the fastest (what Ctx::tune
// does for the operators of fr_setup); for an operator that does not fit shared memory, also time the other form of the plan
// (resident row blocks / streamed operator) and keep the faster one.  Results do not depend on the choice (panel.cuh).
// FRB_AUTOTUNE=0 skips it.
namespace {

template <typename T>
struct TuneScratch {
  T *B = nullptr, *C = nullptr;
  long long N = 0;
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  bool init(int M, int K) {
    // columns: 320 MB of B and C, a multiple of 5 * 128
    N = (long long)(320e6 / ((double)(M + K) * sizeof(T)));
    N = std::max<long long>(640, N / 640 * 640);
    if (cudaMalloc(&B, (size_t)K * N * sizeof(T)) != cudaSuccess) return false;
    if (cudaMalloc(&C, (size_t)M * N * sizeof(T)) != cudaSuccess) return false;
    cudaMemset(B, 0, (size_t)K * N * sizeof(T));
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    return true;
  }
  ~TuneScratch() {
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    if (B) cudaFree(B);
    if (C) cudaFree(C);
  }
  template <typename F>
  float time(F &&run) {
    float best = 1e30f;
    for (int rep = 0; rep < 4; ++rep) {
      cudaEventRecord(e0, 0);
      run();
      cudaEventRecord(e1, 0);
      cudaEventSynchronize(e1);
      float ms = 0;
      cudaEventElapsedTime(&ms, e0, e1);
      if (rep > 0) best = std::min(best, ms);
    }
    return best;
  }
};

// geometry candidates of the plan's (first) panel operator; the other row blocks take the winner's index
template <typename T>
void tune_geometry(GemmPlan<T> &p, const double *A_host, double drop_rel, TuneScratch<T> &sc) {
  PanelOp<T> *cur = p.pop ? p.pop : p.part[0];
  const int M = cur->M, K = p.K, stream = cur->streamed();
  auto time_op = [&](const PanelOp<T> &op) {
    return sc.time([&] { panel_gemm_run(op, sc.N, T(1), sc.B, sc.N, 0, T(0), sc.C, sc.N, 0, 1, (cudaStream_t)0); });
  };
  float bt = time_op(*cur);
  int bestk = 0;
  const int ncand = getenv("FRB_TUNE_CANDS") ? std::max(1, atoi(getenv("FRB_TUNE_CANDS"))) : 14;
  for (int k = 1; k < ncand; ++k) {
    PanelOp<T> op;
    if (!panel_gemm_build(op, M, K, A_host, k, drop_rel, stream)) break;
    const float t = time_op(op);
    if (t < bt) {
      panel_op_free(*cur);
      *cur = op;
      bt = t;
      bestk = k;
    } else {
      panel_op_free(op);
    }
  }
  for (int i = 1; i < p.nparts && bestk > 0; ++i) {
    PanelOp<T> op;
    if (panel_gemm_build(op, p.part[i]->M, K, A_host + (size_t)p.part_row0[i] * K, bestk, drop_rel, stream)) {
      panel_op_free(*p.part[i]);
      *p.part[i] = op;
    }
  }
}

}  // namespace

template <typename T>
void gemm_plan_tune(GemmPlan<T> &p, const double *A_host, double drop_rel) {
  const char *env = getenv("FRB_AUTOTUNE");
  if (env && atoi(env) == 0) return;
  if (!p.pop && p.nparts == 0) return;
  TuneScratch<T> sc;
  if (!sc.init(p.M, p.K)) return;
  tune_geometry(p, A_host, drop_rel, sc);
  const int cur_stream = (p.pop ? p.pop : p.part[0])->streamed();
  if ((p.pop && !cur_stream) || getenv("FRB_GEMM_STREAM")) return;   // the whole image is resident, or the form is forced
  GemmPlan<T> q;
  if (!plan_variant(q, p.M, p.K, A_host, drop_rel, 1 - cur_stream, 1)) return;
  tune_geometry(q, A_host, drop_rel, sc);
  auto time_plan = [&](const GemmPlan<T> &g) {
    return sc.time([&] { gemm_run(g, sc.N, T(1), sc.B, sc.N, 0, T(0), sc.C, sc.N, 0, 1, (cudaStream_t)0); });
  };
  if (time_plan(q) < time_plan(p)) std::swap(p, q);
  gemm_plan_free(q);
}

template <typename T>
void gemm_plan_free(GemmPlan<T> &p) {
  if (p.At) cudaFree(p.At);
  p.At = nullptr;
  if (p.pop) {
    panel_op_free(*p.pop);
    delete p.pop;
    p.pop = nullptr;
  }
  for (int i = 0; i < p.nparts; ++i) {
    panel_op_free(*p.part[i]);
    delete p.part[i];
    p.part[i] = nullptr;
  }
  p.nparts = 0;
}

template <typename T>
int gemm_run(const GemmPlan<T> &p, long long N, T c1, const T *B, long long ldb, long long bstrideB, T c2, T *C,
             long long ldc, long long bstrideC, int nbatch, cudaStream_t s) {
  constexpr int CT = VecT<T>::CT;
  if (N <= 0 || nbatch <= 0) return 0;
  FR_REQUIRE(ldb >= N && ldc >= N, "gemm: leading dimensions must be >= N");
  FR_REQUIRE((ldb * sizeof(T)) % 16 == 0 && (ldc * sizeof(T)) % 16 == 0 && ((uintptr_t)B % 16) == 0 &&
                 ((uintptr_t)C % 16) == 0 && (bstrideB * sizeof(T)) % 16 == 0 && (bstrideC * sizeof(T)) % 16 == 0,
             "gemm: B and C rows must be 16-byte aligned");
  if (p.pop) {
    panel_gemm_run(*p.pop, N, c1, B, ldb, bstrideB, c2, C, ldc, bstrideC, nbatch, s);
    return 1;
  }
  if (p.nparts > 0) {
    for (int i = 0; i < p.nparts; ++i)
      panel_gemm_run(*p.part[i], N, c1, B, ldb, bstrideB, c2, C + (long long)p.part_row0[i] * ldc, ldc, bstrideC, nbatch, s);
    return p.nparts;
  }
  GemmArgs<T> a;
  a.M = p.M;
  a.K = p.K;
  a.nchunks = (p.K + KC - 1) / KC;
  a.nrb = p.nrb;
  a.nbatch = nbatch;
  a.N = N;
  a.ntn = (N + 32 * CT - 1) / (32 * CT);
  a.At = p.At;
  a.B = B;
  a.C = C;
  a.ldb = ldb;
  a.ldc = ldc;
  a.bsB = bstrideB;
  a.bsC = bstrideC;
  a.c1 = c1;
  a.c2 = c2;
  const int grid = 0;
  switch (p.TY) {
    case 4: launch_ty<T, 4>(p, a, grid, s); break;
    case 6: launch_ty<T, 6>(p, a, grid, s); break;
    case 8: launch_ty<T, 8>(p, a, grid, s); break;
    default: throw Error{FR_EINVAL, "gemm: bad TY"};
  }
  return 1;
}

// ---------------------------------------------------------------------------- fr_gemm_static (include/frb200.h)
// The one-shot product for callers that must not allocate device memory (inside a serving loop, under a harness that forbids
// cudaMalloc).  fr_gemm uploads the packed operator into a buffer it allocates and frees; here that buffer is a file-scope
// device array of FR_GEMM_STATIC_MAX_BYTES, which every device that loads the library holds until the process exits.  The
// product runs on the streaming kernel k_gemm above (its operator image is one flat array; the panel kernels' images are several
// arrays sized by the packing).  No cudaMalloc / cudaFree and no allocating library routine on this path.
namespace {

static __device__ __align__(256) unsigned char g_static_op[FR_GEMM_STATIC_MAX_BYTES];

// In host code `g_static_op` is the host-side shadow of the symbol, not a device address: the address a kernel may use comes
// from cudaGetSymbolAddress, asked once per device with that device current.
constexpr int kMaxDevices = 64;
std::mutex g_static_mu;                       // guards g_static_addr and serialises the calls (they share the array)
void *g_static_addr[kMaxDevices] = {};

void *static_op_address() {
  int dev = 0;
  FR_CUDA_TRY(cudaGetDevice(&dev));
  FR_REQUIRE(dev >= 0 && dev < kMaxDevices, "fr_gemm_static: device ordinal out of range");
  if (!g_static_addr[dev]) {
    void *p = nullptr;
    FR_CUDA_TRY(cudaGetSymbolAddress(&p, g_static_op));
    FR_REQUIRE(p != nullptr, "fr_gemm_static: cudaGetSymbolAddress returned NULL");
    g_static_addr[dev] = p;
  }
  return g_static_addr[dev];
}

// thread grid and row blocks of k_gemm for an M x K operator (the choice gemm_plan_build makes for its streaming path); returns
// the number of entries of the packed image [nrb][Kpad][TY*MT]
template <typename T>
size_t static_layout(GemmPlan<T> &p, int M, int K) {
  constexpr int CT = VecT<T>::CT;
  p.M = M;
  p.K = K;
  double best = 1e300;
  for (int ty : {4, 6, 8})
    for (int mt = 2; mt <= 16; mt += 2) {
      const int tile = ty * mt;
      const int nrb = (M + tile - 1) / tile;
      const double score = (double)nrb * tile * (1.0 + 0.15 * (nrb - 1)) - 1e-3 * ty;
      if (score < best) {
        best = score;
        p.TY = ty;
        p.MT = mt;
        p.nrb = nrb;
      }
    }
  const int MTILE = p.TY * p.MT;
  const int Kpad = (K + KC - 1) / KC * KC;
  const size_t slab = (size_t)Kpad * MTILE * sizeof(T);
  p.resident = slab <= 96 * 1024;
  p.smem = (size_t)NSTAGE * KC * 32 * CT * sizeof(T) + (p.resident ? slab : (size_t)NSTAGE * KC * MTILE * sizeof(T));
  return (size_t)p.nrb * Kpad * MTILE;
}

}  // namespace

template <typename T>
void gemm_static_run(int M, int K, long long N, T c1, const double *A_host, const T *B, long long ldb, T c2, T *C, long long ldc,
                     cudaStream_t s) {
  FR_REQUIRE(M > 0 && K > 0 && A_host, "fr_gemm_static: M, K must be positive and A non-NULL");
  FR_REQUIRE(N >= 0 && B && C, "fr_gemm_static: N must be >= 0 and B, C non-NULL");
  GemmPlan<T> p;
  const size_t n = static_layout(p, M, K);
  if (n * sizeof(T) > (size_t)FR_GEMM_STATIC_MAX_BYTES)
    throw Error{FR_EINVAL, "fr_gemm_static: the packed " + std::to_string(M) + " x " + std::to_string(K) + " operator takes " +
                               std::to_string(n * sizeof(T)) + " bytes, more than FR_GEMM_STATIC_MAX_BYTES = " +
                               std::to_string((size_t)FR_GEMM_STATIC_MAX_BYTES) + " (use fr_gemm or fr_gemm_plan_*)"};
  // the whole image is written on every call, zero padding included: nothing of the previous call's operator survives
  std::vector<T> At(n, T(0));
  const int MTILE = p.TY * p.MT, Kpad = (K + KC - 1) / KC * KC;
  for (int m = 0; m < M; ++m)
    for (int k = 0; k < K; ++k) {
      const double v = A_host[(size_t)m * K + k];
      FR_REQUIRE(v == v && v - v == 0.0, "fr_gemm_static: operator contains non-finite entries");
      At[((size_t)(m / MTILE) * Kpad + k) * MTILE + m % MTILE] = (T)v;
    }
  std::lock_guard<std::mutex> lock(g_static_mu);
  p.At = static_cast<T *>(static_op_address());
  FR_CUDA_TRY(cudaMemcpyAsync(p.At, At.data(), n * sizeof(T), cudaMemcpyHostToDevice, s));
  gemm_run(p, N, c1, B, ldb, 0, c2, C, ldc, 0, 1, s);
  // the next call overwrites the array and `At` goes out of scope: wait for the copy and the product
  FR_CUDA_TRY(cudaStreamSynchronize(s));
}

template void gemm_static_run<double>(int, int, long long, double, const double *, const double *, long long, double, double *,
                                      long long, cudaStream_t);
template void gemm_static_run<float>(int, int, long long, float, const double *, const float *, long long, float, float *, long long,
                                     cudaStream_t);

template void gemm_plan_build<double>(GemmPlan<double> &, int, int, const double *, double);
template void gemm_plan_build<float>(GemmPlan<float> &, int, int, const double *, double);
template void gemm_plan_tune<double>(GemmPlan<double> &, const double *, double);
template void gemm_plan_tune<float>(GemmPlan<float> &, const double *, double);
template void gemm_plan_free<double>(GemmPlan<double> &);
template void gemm_plan_free<float>(GemmPlan<float> &);
template int gemm_run<double>(const GemmPlan<double> &, long long, double, const double *, long long, long long, double,
                              double *, long long, long long, int, cudaStream_t);
template int gemm_run<float>(const GemmPlan<float> &, long long, float, const float *, long long, long long, float,
                             float *, long long, long long, int, cudaStream_t);

}  // namespace frb
