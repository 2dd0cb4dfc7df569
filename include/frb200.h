/* frb200.h -- C ABI of the B200-native flux-reconstruction hot path.
 *
 * What is computed: one evaluation of the flux-reconstruction right-hand side of the 3-D compressible
 * Euler / Navier-Stokes equations on mixed prism / tetrahedron grids, and Runge-Kutta steps built on it.
 * The paper (arXiv 1409.0405, text in /root/reference/PAPER.md, cited as P:line) states the shape of that
 * computation: "The majority of operations within an FR time-step can be cast as matrix multiplications of
 * the form C <- c1 A B + c2 C [eq. 1] where ... A is a constant operator matrix, and B and C are row-major
 * state matrices", "All other operations ... are point-wise, concerning themselves solely with data
 * at an individual solution/flux point"; systems, element types, steppers and precisions: Table 1
 * (P:23); compressible Navier-Stokes with constant viscosity, DG scheme, Rusanov Riemann solver, RK45[2R+]
 * (P:116); boundary-condition types of the cylinder case.  The formulas the paper defers to its
 * references are fixed in DESIGN.md ("Readings", R1-R22) and SURVEY.md Appendix A / C.
 *
 * General rules
 *   - Every function returns fr_status (FR_OK = 0) unless stated; no exceptions, no abort, nothing printed.
 *   - "HOST" pointers are ordinary host memory, borrowed for the duration of the call only; the library
 *     copies what it needs.  "DEVICE" pointers are CUDA device memory owned by the caller (e.g. a torch
 *     tensor's data_ptr()).  All host-side floating point inputs are FP64; with FR_F32 the library rounds
 *     them once (round-to-nearest-even) and computes in FP32 (reading R15).
 *   - State layout of one element type on the device: [nupts][5][ld] in the chosen precision, element
 *     index fastest ("row-major state matrix" of P:39 with column = v*ld + e, reading R5); ld >= neles is
 *     the padded leading dimension reported by fr_state_layout (ld * sizeof(real) is a multiple of 128).
 *     Padding columns are ignored on input and written as zero on output.
 *   - All work is enqueued on the CUDA stream given in fr_config (asynchronous); fr_sync waits and
 *     surfaces asynchronous errors.  Same inputs give bitwise-identical outputs (no atomics).
 *   - One context per host thread; calls on one context must be serialised by the caller.
 *   - There is no CPU fallback: without a usable CUDA device fr_setup / fr_gemm return FR_ECUDA.
 */
#ifndef FRB200_H
#define FRB200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct fr_ctx fr_ctx;

typedef enum { FR_OK = 0, FR_EINVAL = 1, FR_ENOMEM = 2, FR_ECUDA = 3, FR_ESTATE = 4, FR_EUNSUPPORTED = 5 } fr_status;
typedef enum { FR_F32 = 4, FR_F64 = 8 } fr_prec;                 /* P:23 "Precisions: Single, Double" */
typedef enum { FR_EULER = 0, FR_NAVIER_STOKES = 1 } fr_system;   /* P:23 "Governing Systems" */
typedef enum { FR_TET = 0, FR_PRI = 1, FR_HEX = 2 } fr_etype;    /* P:23 (3-D element types of Table 1) */
typedef enum { FR_RK4 = 0, FR_RK45_2R = 1, FR_EULER1 = 2 } fr_stepper;   /* P:23 "Time Steppers: Euler, RK4, RK45"; P:116 RK45[2R+] */
typedef enum { FR_BC_NOSLIP_ISOTHERMAL_WALL = 0, FR_BC_CHAR_RIEMANN_INV = 1 } fr_bctype;
typedef enum { FR_MODE_FUSED = 0, FR_MODE_UNFUSED = 1 } fr_mode; /* kernel chain: fused (default) or one kernel per step */

/* One per element type present in the mesh.  All pointers HOST, FP64, row-major, borrowed.
 * Operators (constant per element type and order): the "applied" operators of SURVEY 8 / A.4,
 *   M0   [nfpts][nupts]      solution -> flux points ("volume-to-surface interpolation", Table 2)
 *   M132 [nupts][3*nupts]    = M1 - M3*M2, divergence of the transformed flux minus the lifted interior normal flux;
 *                            column = alpha*nupts + nu
 *   M3   [nupts][nfpts]      lift of the common normal flux (DG correction functions, "A DG scheme")
 *   M460 [3*nupts][nupts]    = M4 - M6*M0, reference gradient minus lifted interior values; row = alpha*nupts + rho
 *   M6   [3*nupts][nfpts]    lift of the common solution into the gradient
 * M460 and M6 may be NULL for FR_EULER. */
typedef struct {
  fr_etype etype;
  int32_t order, nupts, nfpts;
  int64_t neles;
  int32_t affine;        /* 1: metric terms constant per element (smats [3][3][neles], rcpdjac [neles]) */
  const double *M0, *M132, *M3, *M460, *M6;
  const double *smats;   /* [3 alpha][3 i][nupts][neles]  S = |J| * d(xref_alpha)/d(x_i);  [3][3][neles] if affine */
  const double *rcpdjac; /* [nupts][neles]  1/|J|;  [neles] if affine */
} fr_eles_desc;

/* Interior and periodic flux-point pairs.  The L/R designation is the caller's and is binding (the LDG
 * common values are not symmetric, reading R9).  Every (et, ele, fpt) of the mesh must appear exactly once
 * across the pairs and the boundary lists, otherwise fr_setup returns FR_EINVAL. */
typedef struct {
  int64_t npairs;
  const int32_t *l_et, *l_fpt;  /* index into eles[], flux point sigma in [0, nfpts) */
  const int64_t *l_ele;
  const int32_t *r_et, *r_fpt;
  const int64_t *r_ele;
  const double *nl;             /* [3][npairs] unit physical normal, outward from L */
  const double *magl, *magr;    /* [npairs] |S^T n_ref| on each side (not equal in general) */
} fr_iface_desc;

/* Boundary flux points of one boundary condition.  params:
 *   FR_BC_NOSLIP_ISOTHERMAL_WALL: params[0] = c_v * T_wall
 *   FR_BC_CHAR_RIEMANN_INV      : params[0..4] = rho_inf, vx_inf, vy_inf, vz_inf, p_inf */
typedef struct {
  fr_bctype type;
  int64_t nfpts;
  const int32_t *et, *fpt;
  const int64_t *ele;
  const double *n;              /* [3][nfpts] unit outward normal */
  const double *mag;            /* [nfpts] */
  double params[8];
} fr_bc_desc;

/* Domain decomposition (section 2.5: ranks exchange interface data).  A flux-point pair cut by the partition
 * names its remote side in fr_iface_desc as element type `netypes` (one past the rank's own types), flux point 0, element g:
 * "ghost" g, 0 <= g < nghost, each referenced by exactly one pair.  (et, fpt, ele)[g] is the OWN flux point of that same pair,
 * whose interpolated state (and, for Navier-Stokes, gradient) the peer needs: send entry g and ghost g belong to one cut pair,
 * so a rank's ghosts of a peer and what it sends to that peer are the same index range, ordered alike on both ranks.
 * All pointers HOST, borrowed for fr_setup. */
typedef struct {
  int64_t nghost;
  const int32_t *et, *fpt;
  const int64_t *ele;
} fr_halo_desc;

typedef struct {
  fr_system system;
  fr_prec prec;
  fr_stepper stepper;
  fr_mode mode;
  double gamma, mu, prandtl;    /* ideal gas; constant viscosity; Pr */
  double ldg_beta, ldg_tau;     /* LDG upwinding and penalty parameters (reading R9) */
  int32_t netypes;
  const fr_eles_desc *eles;     /* [netypes] */
  const fr_iface_desc *ifaces;  /* one descriptor */
  int32_t nbcs;
  const fr_bc_desc *bcs;        /* [nbcs], may be NULL if nbcs == 0 */
  void *cuda_stream;            /* cudaStream_t; NULL = default stream */
  const fr_halo_desc *halo;     /* NULL: the whole domain is on this GPU */
} fr_config;

/* Validate, copy to the device, build the interface views.  On failure *out = NULL and
 * fr_global_error() describes the problem.  Ownership of every input stays with the caller. */
fr_status fr_setup(const fr_config *cfg, fr_ctx **out);

/* Device layout of element type `et`: leading dimension (elements) and bytes of one state array. */
fr_status fr_state_layout(const fr_ctx *ctx, int32_t et, int64_t *ld, int64_t *nbytes);

/* dudt = RHS(u) -- steps S1..S9 of SURVEY 8(a).  u_dev / dudt_dev: arrays [netypes] of DEVICE
 * pointers in the fr_state_layout layout and the context's precision; u is not modified; dudt must not
 * alias u.  Asynchronous on the context's stream. */
fr_status fr_rhs(fr_ctx *ctx, const void *const *u_dev, void *const *dudt_dev);

/* Host [nupts][5][neles] FP64 <-> internal solution register (rounds if FR_F32).  Synchronous. */
fr_status fr_set_state(fr_ctx *ctx, const double *const *u_host);
fr_status fr_get_state(fr_ctx *ctx, double *const *u_host);

/* Advance the internal state by one step of the configured stepper with step dt (forward Euler, RK4: P:23; RK45[2R+]:
 * P:116, coefficients reading R12; fixed dt, no error control).  The stage update is fused into the last
 * kernel of each RHS (S10).  The kernel sequence of a step is captured once into a CUDA graph and
 * replayed.  Asynchronous.  fr_rk_run = nsteps calls of fr_rk_step without host synchronisation. */
fr_status fr_rk_step(fr_ctx *ctx, double dt);
fr_status fr_rk_run(fr_ctx *ctx, double dt, int64_t nsteps);

/* Adaptive RK45[2R+] (the embedded pair P:116 names, reading R12 for b-hat, R25 for the norm and the
 * controller): advance the internal state from t0 to t1 with step-size control.  FR_RK45_2R contexts only.
 * Every attempt uses dt = min(dt, t1 - t) and evaluates
 *   E = dt sum_i (b_i - bhat_i) K_i,   err = sqrt( mean over solution points and variables of (E / (atol + rtol max(|u_n|, |u_n+1|)))^2 );
 * it is accepted iff err <= 1 (otherwise the state is restored); after every attempt
 *   dt <- dt * clip(0.8 err^(-0.7/4) err_prev^(0.4/4), 0.3, 2.5),  err_prev = error of the last accepted step (1 initially),
 * a non-finite err counting as a rejection with factor 0.3.  The five stages, the error accumulation (three extra registers: E,
 * u_n, and the stage register kept after the last stage) and a deterministic two-pass reduction of the norm run as one CUDA
 * graph per attempt; the accept / reject decision and the controller run on the host in FP64 after reading back one scalar.
 * stats (HOST, may be NULL): accepted, rejected, t reached (== t1 unless max_attempts ran out: FR_ESTATE then), dt proposed for
 * the next step.  dt_hist / err_hist (HOST, may be NULL, capacity hist_cap): dt tried and err of every attempt, in order.
 * Synchronous. */
typedef struct {
  int64_t accepted, rejected;
  double t, dt_next;
} fr_adapt_stats;
fr_status fr_rk_adaptive_run(fr_ctx *ctx, double t0, double t1, double dt_init, double atol, double rtol, int64_t max_attempts,
                             fr_adapt_stats *stats, double *dt_hist, double *err_hist, int64_t hist_cap);

/* Waits for the stream; returns FR_ECUDA if any asynchronous error occurred. */
fr_status fr_sync(fr_ctx *ctx);

/* Number of kernels this context has launched (graph replays count their kernel nodes). */
int64_t fr_launch_count(const fr_ctx *ctx);

/* Time, with CUDA events on the context's stream, `reps` evaluations of the RHS of the internal state and
 * return the mean milliseconds per kernel group: ms[0] operator products (S1,S3,S5,S8 incl. fused point-wise
 * work), ms[1] point-wise solution-point kernels, ms[2] interface / boundary kernels, ms[3] total.
 * Synchronous; measurement aid for BASELINE.json configs[4] ("per-kernel time breakdown"). */
fr_status fr_profile_rhs(fr_ctx *ctx, int32_t reps, double ms[4]);

/* Per-kernel version of fr_profile_rhs: one entry per kernel (or kernel pair of one step) of a single RHS
 * evaluation, in launch order.  name = "<tet|pri>:<step>" or "<step>" for the interface kernels; ms = mean CUDA-event
 * time; alg_bytes / flops = ALGORITHMIC traffic and arithmetic of that launch (every operand read or written once;
 * 2 flops per NON-ZERO operator entry and column for the products on the panel kernels -- structural zeros of the prism
 * operators are skipped at set-up and not counted -- dense 2*M*K*N on the unfused fall-back).
 * Writes min(*n, cap)
 * entries and sets *n to the number of kernels. */
typedef struct {
  char name[48];
  double ms, alg_bytes, flops;
  int32_t category;   /* 0 operator product, 1 point-wise at solution points, 2 interface / boundary */
} fr_kernel_stat;
fr_status fr_profile_kernels(fr_ctx *ctx, int32_t reps, fr_kernel_stat *out, int32_t cap, int32_t *n);
/* The same for the right-hand side AS A RUNGE-KUTTA STAGE runs it (the variant fr_rk_step replays: S10 of SURVEY 8(a), the
 * stage update X <- X + c1 K, Y <- X + c2 K, fused into the last kernel of each type, with both coefficients zero here so the
 * internal state is unchanged). */
fr_status fr_profile_stage_kernels(fr_ctx *ctx, int32_t reps, fr_kernel_stat *out, int32_t cap, int32_t *n);

/* Failure detection off the hot path: counts the non-finite entries (NaN / Inf) of the internal solution register,
 * padding columns excluded.  Synchronous. */
fr_status fr_check_finite(fr_ctx *ctx, int64_t *n_nonfinite);

/* The launch plan fr_setup chose (packing, warp grid, panel width, ring depth per operator), one line per operator, as a
 * NUL-terminated string of at most cap - 1 characters.  Results never depend on it (bit-identical for every plan). */
fr_status fr_plan_describe(const fr_ctx *ctx, char *buf, int64_t cap);

/* Partitioned right-hand side (fr_config.halo): fr_rhs cut at its two exchange points.
 *   phase 0: S1 (U_f = M0 U), then the own U_f at the cut flux points is packed into the U send buffer;
 *   phase 1: the received U_f is unpacked into the ghost flux points; S2..S5; the own G_f is packed (Navier-Stokes);
 *   phase 2: the received G_f is unpacked (Navier-Stokes); S7, S6, S8..S10 -> dudt.
 * Between the phases the caller moves send buffers into the peers' receive buffers (fr_halo_buffers) on the context's stream --
 * NCCL send/recv over NVLink through torch.distributed in paper_1409_0405_b200/halo.py.  u_dev / dudt_dev as for fr_rhs (dudt_dev
 * may be NULL in phases 0 and 1).  Without a halo descriptor phases 0, 1, 2 in a row are exactly fr_rhs. */
fr_status fr_rhs_phase(fr_ctx *ctx, int32_t phase, const void *const *u_dev, void *const *dudt_dev);
/* The same for stage `stage` (0-based) of a Runge-Kutta step of size dt on the internal state (S10 fused into phase 2). */
fr_status fr_rk_stage_phase(fr_ctx *ctx, double dt, int32_t stage, int32_t phase);
/* Device buffers of the exchange: which = 0 the interpolated state (V = 5 values per flux point), 1 its gradient (V = 15).
 * Layout of both buffers: for the flux points [start, start + count) exchanged with one peer, value v of flux point start + j
 * is element V*start + v*count + j -- one contiguous message of V*count values per peer.  *nvalues = V * nghost.
 * Owned by the context. */
fr_status fr_halo_buffers(fr_ctx *ctx, int32_t which, void **send_dev, void **recv_dev, int64_t *nvalues);
/* The peer segmentation the buffers use: (start, count) per peer, in ghost order; must cover [0, nghost) (FR_EINVAL otherwise). */
fr_status fr_halo_set_peers(fr_ctx *ctx, int32_t npeers, const int64_t *start, const int64_t *count);

/* End-to-end step on HOST buffers: copies u_host[t] (HOST, fr_state_layout layout and the context's precision,
 * ideally pinned) into the solution register, advances one step of size dt, copies the new state back into the
 * same buffers and waits.  The host<->device copies are part of the call. */
fr_status fr_rk_step_host(fr_ctx *ctx, double dt, void *const *u_host);

const char *fr_last_error(const fr_ctx *ctx);   /* owned by ctx, valid until the next call on it */
const char *fr_global_error(void);              /* message of the last failed fr_setup / fr_gemm on this thread */
void fr_destroy(fr_ctx *ctx);

/* Stand-alone operator product C <- c1*A*B + c2*C (eq. 1) for BASELINE.json configs[3].
 * A: HOST FP64 [M][K] row-major (rounded to `prec`); B: DEVICE [K][ldb], C: DEVICE [M][ldc] in `prec`,
 * N columns used; ldb, ldc >= N with ld*sizeof(real) a multiple of 16 and 16-byte aligned bases
 * (FR_EINVAL otherwise).  If c2 == 0, C is not read.  Runs on `cuda_stream` and returns after the product has
 * completed (A is uploaded and released inside the call; use fr_gemm_plan_* to keep A resident). */
fr_status fr_gemm(int32_t M, int32_t K, int64_t N, double c1, const double *A_host, const void *B_dev, int64_t ldb,
                  double c2, void *C_dev, int64_t ldc, fr_prec prec, void *cuda_stream);

/* fr_gemm for callers that must not allocate device memory (a serving loop, a harness that forbids cudaMalloc): the same
 * product (eq. 1), arguments, layouts, alignment rules and completion semantics as fr_gemm, but the device copy of the
 * packed operator lives in a file-scope device array of FR_GEMM_STATIC_MAX_BYTES that every GPU holding the library keeps until
 * the process exits; the call makes no cudaMalloc / cudaFree and calls no allocating library routine.  An operator whose packed
 * image (rows and K padded to the kernel's tiles) exceeds the array is rejected with FR_EINVAL and a message naming both sizes
 * (e.g. FP64 192 x 64 = 98 KB fits; 343 x 343 does not: use fr_gemm or a plan).  The product runs on the streaming kernel
 * (FFMA / DFMA register tiles, gemm.cu), so its results agree with fr_gemm's to rounding, not bit for bit.
 * All calls on one device share the array and each rewrites all of it (zero padding included), so nothing of an earlier call's
 * operator is ever read.  The library serialises the calls of one process with a host lock held until the product has
 * completed; work that reads or writes the array outside that lock while a call is in flight would race with it. */
#define FR_GEMM_STATIC_MAX_BYTES (512 * 1024)
fr_status fr_gemm_static(int32_t M, int32_t K, int64_t N, double c1, const double *A_host, const void *B_dev, int64_t ldb,
                         double c2, void *C_dev, int64_t ldc, fr_prec prec, void *cuda_stream);

/* The same product with A uploaded once: plan -> run (asynchronous, launch only) -> destroy. */
typedef struct fr_gemm_plan fr_gemm_plan;
fr_status fr_gemm_plan_create(int32_t M, int32_t K, const double *A_host, fr_prec prec, fr_gemm_plan **out);
fr_status fr_gemm_plan_run(fr_gemm_plan *plan, int64_t N, double c1, const void *B_dev, int64_t ldb, double c2,
                           void *C_dev, int64_t ldc, void *cuda_stream);
/* How the plan runs, one line per kernel launch: precision, rows of A it covers, packing ("dense", "k-lists", "dense, streamed" = an
 * operator too large for shared memory whose packed blocks travel through the TMA ring with the chunks of B; otherwise such
 * operators run as row blocks of A, one launch each), warp grid, panel width, chunk count and ring depth.  fr_gemm_plan_create
 * times the candidate forms and keeps the fastest; every form gives bit-identical results.  NUL-terminated, at most cap - 1
 * characters. */
fr_status fr_gemm_plan_describe(const fr_gemm_plan *plan, char *buf, int64_t cap);
void fr_gemm_plan_destroy(fr_gemm_plan *plan);

/* Measured device peaks used as roofline denominators: register-resident FMA
 * chains (TFLOP/s, FP64 and FP32) and a device-to-device copy (GB/s, read+write bytes).  Synchronous. */
fr_status fr_probe_peaks(double *fp64_tflops, double *fp32_tflops, double *copy_gbs);
/* The FP64 tensor pipe (mma.sync.m8n8k4.f64, what the FP64 operator products run on): TFLOP/s of
 * register-resident chains, 512 flops per warp instruction.  The denominator of compute-bound FP64 roofline fractions. */
fr_status fr_probe_dmma(double *fp64_tensor_tflops);

/* The FP32 alternatives weighed in DESIGN.md section 6, as register-resident chains (TFLOP/s): packed fma.rn.f32x2 (FFMA2: what the
 * FP32 operator products use); FFMA and FFMA2 chains with eight integer multiply-adds beside every sixteen FMAs (the issue slots that
 * address arithmetic costs a multiply loop); the legacy TF32 tensor path mma.sync.m16n8k8 (dense rate; an error-compensated 3xTF32
 * product would run at a third of it).  Any pointer may be NULL. */
fr_status fr_probe_fp32_paths(double *ffma2_tflops, double *ffma_mixed_tflops, double *ffma2_mixed_tflops, double *tf32_mma_tflops);

#ifdef __cplusplus
}
#endif
#endif /* FRB200_H */
