// Shared declarations of the frb200 library (host + device).  sm_100a only.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>

#include <string>
#include <vector>

#include "../../include/frb200.h"

#define FR_NVAR 5
#define FR_MAXTYPES 4

namespace frb {

struct Error {
  fr_status st;
  std::string msg;
};

#define FR_CUDA_TRY(expr)                                                                       \
  do {                                                                                          \
    cudaError_t _e = (expr);                                                                    \
    if (_e != cudaSuccess) {                                                                    \
      throw frb::Error{FR_ECUDA, std::string(#expr) + ": " + cudaGetErrorString(_e)};           \
    }                                                                                           \
  } while (0)

#define FR_REQUIRE(cond, msg_)                                                                  \
  do {                                                                                          \
    if (!(cond)) throw frb::Error{FR_EINVAL, std::string(msg_)};                                \
  } while (0)

// Per-type addressing table of the flat flux-point arrays, passed by value to the interface kernels.
// U_f / C / D of type t: [nfpts][5][ld] at ubase[t];  G_f: [3][nfpts][5][ld] at gbase[t].
struct TypeTab {
  long long ubase[FR_MAXTYPES];
  long long gbase[FR_MAXTYPES];
  long long ld[FR_MAXTYPES];
  long long gcomp[FR_MAXTYPES];   // nfpts*5*ld: stride between gradient components in G_f
};

// One side of a flux-point pair: element index and (type << 16 | sigma).
struct PairRec {
  int le, lts, re, rts;
};
struct BndRec {
  int e, ts;
};

template <typename T>
struct PhysParams {
  T gamma, mu, prandtl, beta, tau;
  int ns;
};

// Stage-update coefficients live in device memory so a captured graph needs no re-capture when dt changes.
struct StageCoef {
  double c1, c2;
};

template <typename T>
struct PanelOp;   // panel.cuh: operator packed for the resident-operator panel kernels

template <typename T>
struct GemmPlan {
  int M = 0, K = 0;
  int TY = 0, MT = 0, nrb = 0;   // thread rows, rows per thread, row blocks (M <= nrb*TY*MT)
  int resident = 0;              // whole operator slab kept in shared memory
  int ctas_per_sm = 1;
  size_t smem = 0;
  T *At = nullptr;               // device, [nrb][K][TY*MT], zero padded, transposed operator
  PanelOp<T> *pop = nullptr;     // non-null: the panel kernel serves this operator (At is then unused)
  // operators with too many rows for one CTA: row blocks of A, each its own panel operator, launched one after the other
  // (B is read once per block: these are the compute-bound shapes)
  static constexpr int kMaxParts = 32;
  int nparts = 0;
  PanelOp<T> *part[kMaxParts] = {};
  int part_row0[kMaxParts] = {};
};

// drop_rel: entries with |a| <= drop_rel * max|A| are treated as structural zeros when the operator is packed (reading R24: the FR
// operators handed to fr_setup); the public fr_gemm passes 0 (only exact zeros are skipped)
template <typename T>
void gemm_plan_build(GemmPlan<T> &p, int M, int K, const double *A_host, double drop_rel = 1.4210854715202004e-14);
// times the plan's launch geometries on scratch matrices and keeps the fastest (fr_gemm_plan_create)
template <typename T>
void gemm_plan_tune(GemmPlan<T> &p, const double *A_host, double drop_rel);
template <typename T>
void gemm_plan_free(GemmPlan<T> &p);
// C[b] <- c1 * A * B[b] + c2 * C[b], b < nbatch; returns the number of kernels launched
template <typename T>
int gemm_run(const GemmPlan<T> &p, long long N, T c1, const T *B, long long ldb, long long bstrideB, T c2, T *C,
             long long ldc, long long bstrideC, int nbatch, cudaStream_t s);
// fr_gemm_static: the one-shot product with the packed operator in a file-scope device array (gemm.cu); allocates nothing, synchronous
template <typename T>
void gemm_static_run(int M, int K, long long N, T c1, const double *A_host, const T *B, long long ldb, T c2, T *C, long long ldc,
                     cudaStream_t s);

int device_sm_count();

}  // namespace frb
