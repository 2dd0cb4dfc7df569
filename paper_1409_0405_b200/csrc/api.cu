// C ABI (include/frb200.h): context set-up, device data model, RHS stage driver, Runge-Kutta graphs.
#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <memory>
#include <numeric>

#include <nvtx3/nvToolsExt.h>

#include "kernels.cuh"

namespace frb {

// NVTX range around one step of the right-hand side (SURVEY 5 "tracing"): a no-op unless a tool is attached
struct NvtxRange {
  explicit NvtxRange(const char *name) { nvtxRangePushA(name); }
  ~NvtxRange() { nvtxRangePop(); }
};

static thread_local std::string g_error;

struct CtxBase {
  fr_prec prec;
  std::string err;
  long long launches = 0;
  virtual ~CtxBase() {}
  virtual void state_layout(int et, int64_t *ld, int64_t *nbytes) const = 0;
  virtual void rhs(const void *const *u, void *const *dudt) = 0;
  virtual void set_state(const double *const *u) = 0;
  virtual void get_state(double *const *u) = 0;
  virtual void rk_step(double dt, long long nsteps) = 0;
  virtual void sync() = 0;
  virtual void profile(int reps, double ms[4], fr_kernel_stat *out, int cap, int *n, bool stage = false) = 0;
  virtual long long check_finite() = 0;
  virtual void rhs_phase(int phase, const void *const *u, void *const *dudt) = 0;
  virtual void rk_stage_phase(double dt, int stage, int phase) = 0;
  virtual void halo_buffers(int which, void **send, void **recv, int64_t *n) = 0;
  virtual void halo_set_peers(int npeers, const int64_t *start, const int64_t *count) = 0;
  virtual std::string describe() const = 0;
  virtual void rk_step_host(double dt, void *const *u_host) = 0;
  virtual void rk_adaptive(double t0, double t1, double dt0, double atol, double rtol, long long max_attempts, fr_adapt_stats *st,
                           double *dt_hist, double *err_hist, long long hist_cap) = 0;
};

template <typename T>
struct DevBuf {
  T *p = nullptr;
  size_t n = 0;
  void alloc(size_t count, bool zero = true) {
    n = count;
    if (count == 0) return;
    cudaError_t e = cudaMalloc(&p, count * sizeof(T));
    if (e != cudaSuccess) throw Error{FR_ENOMEM, std::string("cudaMalloc: ") + cudaGetErrorString(e)};
    if (zero) FR_CUDA_TRY(cudaMemset(p, 0, count * sizeof(T)));
  }
  void upload(const std::vector<T> &h) {
    alloc(h.size(), false);
    if (n) FR_CUDA_TRY(cudaMemcpy(p, h.data(), n * sizeof(T), cudaMemcpyHostToDevice));
  }
  ~DevBuf() {
    if (p) cudaFree(p);
  }
  DevBuf() = default;
  DevBuf(const DevBuf &) = delete;
  DevBuf &operator=(const DevBuf &) = delete;
};

enum { CAT_GEMM = 0, CAT_PW = 1, CAT_IFACE = 2 };
constexpr long long kIfaceBlock = 256;  // elements per locality block of the interface pair order

// Per-kernel CUDA-event timeline of one RHS evaluation (measurement aid; never active on the normal path).
struct Timeline {
  std::vector<cudaEvent_t> ev;
  std::vector<int> cat;
  std::vector<std::string> name;
  std::vector<double> bytes, flops;
  cudaStream_t s;
  void mark(int c, const std::string &nm = "", double b = 0, double f = 0) {
    cudaEvent_t e;
    cudaEventCreate(&e);
    cudaEventRecord(e, s);
    ev.push_back(e);
    cat.push_back(c);
    name.push_back(nm);
    bytes.push_back(b);
    flops.push_back(f);
  }
};

template <typename T>
struct FusedPart {
  PanelOp<T> op;
  int r0 = 0, nr = 0;   // solution points r0 .. r0+nr-1
};

// Build a fused operator over `nrows` solution points as 1, 2, ... blocks (a multiple of 8 points each, as even as possible)
// until every block fits the panel kernel.  build(op, r0, nr) -> bool.  Leaves `parts` empty if nothing fits.
template <typename T, typename B>
void build_split(std::vector<FusedPart<T>> &parts, int nrows, B build) {
  for (auto &q : parts) panel_op_free(q.op);
  parts.clear();
  const int maxp = getenv("FRB_NO_ROWSPLIT") ? 1 : 32;
  // FRB_FORCE_SPLIT=n: start at n blocks (parity tests of the row split on operators that would fit in one)
  const int minp = getenv("FRB_FORCE_SPLIT") ? std::max(1, std::min(maxp, atoi(getenv("FRB_FORCE_SPLIT")))) : 1;
  for (int np = minp; np <= maxp; ++np) {
    const int per = np == 1 ? nrows : ((nrows + np - 1) / np + 7) / 8 * 8;
    if (np > 1 && (long long)per * (np - 1) >= nrows) continue;
    bool ok = true;
    for (int r0 = 0; r0 < nrows && ok; r0 += per) {
      FusedPart<T> q;
      q.r0 = r0;
      q.nr = std::min(per, nrows - r0);
      ok = build(q.op, q.r0, q.nr);
      if (ok) parts.push_back(q);
    }
    if (ok) return;
    for (auto &q : parts) panel_op_free(q.op);
    parts.clear();
  }
}

template <typename T>
double parts_density(const std::vector<FusedPart<T>> &parts) {
  double a = 0, b = 0;
  for (auto &q : parts) {
    a += q.op.density * q.nr;
    b += q.nr;
  }
  return b > 0 ? a / b : 1.0;
}

template <typename T>
struct EleData {
  EleView<T> view;
  DevBuf<T> smats, rcpdjac;
  GemmPlan<T> pM0, pM132, pM3, pM460, pM6;
  // fused operators [M132 | M3] and [M460 | M6] (FR_MODE_FUSED); more than one entry = blocks of solution points, launched one
  // after the other, for operators with more rows than one CTA's accumulators hold (e.g. hexahedra at p = 4)
  std::vector<FusedPart<T>> pDiv, pGrad;
  DevBuf<T> X, Y, ACC;   // solution register, stage input, RK4 accumulator
  DevBuf<T> E, U0;       // adaptive RK45: error register, state at the start of the attempt (allocated on first use)
  DevBuf<T> grad;        // [3][nupts][5][ld]: G~ -> G -> F~ (S6 in place)
  DevBuf<T> R;           // [nupts][5][ld]
  ~EleData() {
    gemm_plan_free(pM0);
    gemm_plan_free(pM132);
    gemm_plan_free(pM3);
    gemm_plan_free(pM460);
    gemm_plan_free(pM6);
    for (auto &q : pDiv) panel_op_free(q.op);
    for (auto &q : pGrad) panel_op_free(q.op);
  }
};

template <typename T>
struct BndData {
  BndView<T> view;
  DevBuf<BndRec> recs;
  DevBuf<T> nrm, mag;
};

template <typename T>
struct Ctx : CtxBase {
  fr_system system;
  fr_stepper stepper;
  fr_mode mode;
  PhysParams<T> ph;
  cudaStream_t stream = nullptr;
  bool own_stream = false;
  int nt = 0;
  std::vector<std::unique_ptr<EleData<T>>> el;
  const char *tname[FR_MAXTYPES] = {"t0", "t1", "t2", "t3"};
  TypeTab tt;
  DevBuf<T> uf, cf, gf;
  IfaceView<T> iv;
  DevBuf<PairRec> pairs;
  DevBuf<T> nl, magl, magr;
  std::vector<std::unique_ptr<BndData<T>>> bnd;
  DevBuf<StageCoef> coef;
  StageCoef *coef_host = nullptr;   // pinned
  double coef_dt = std::nan("");
  int jump = 0;                     // S2 stores C - U_f and the fused gradient operator is [M4 | M6] (all types fused)
  cudaGraphExec_t graph = nullptr;
  int graph_kernels = 0;
  cudaGraphExec_t graph_adapt = nullptr;   // one attempt of the adaptive stepper: save, 5 stages + error register, norm
  int graph_adapt_kernels = 0;
  DevBuf<double> err_partial, err_dev;      // [nt * rk_err_blocks()], [1 + 2]: sum of squares, then {atol, rtol}
  double *err_host = nullptr;               // pinned: [0] sum of squares read back, [1..2] staging of {atol, rtol}
  double tol_set[2] = {-1.0, -1.0};
  // domain decomposition (fr_config.halo): the remote sides of cut pairs live in a ghost pseudo type (index nt) of the flat
  // flux-point arrays; own values at the cut flux points travel through the send / receive buffers
  long long nghost = 0;
  HaloView hv{};
  DevBuf<long long> h_offu, h_offg, h_ld, h_gcomp, h_pstart, h_pcnt, h_pj;
  DevBuf<T> h_send[2], h_recv[2];
  int cmask = 0;                            // phases that run one branch per element type (run_rhs; FRB_CONCURRENT=mask, 0: one stream)
  std::vector<cudaStream_t> aux;
  std::vector<cudaEvent_t> ev_type;
  cudaEvent_t ev_main[3] = {nullptr, nullptr, nullptr};

  ~Ctx() override {
    for (auto q : aux) cudaStreamDestroy(q);
    for (auto e : ev_type) cudaEventDestroy(e);
    for (auto e : ev_main)
      if (e) cudaEventDestroy(e);
    if (graph) cudaGraphExecDestroy(graph);
    if (graph_adapt) cudaGraphExecDestroy(graph_adapt);
    if (coef_host) cudaFreeHost(coef_host);
    if (err_host) cudaFreeHost(err_host);
    if (own_stream && stream) cudaStreamDestroy(stream);
  }

  // ------------------------------------------------------------------ set-up
  void setup(const fr_config *c) {
    prec = c->prec;
    system = c->system;
    stepper = c->stepper;
    mode = c->mode;
    stream = (cudaStream_t)c->cuda_stream;
    if (getenv("FRB_CONCURRENT")) cmask = atoi(getenv("FRB_CONCURRENT")) & 15;
    if (!stream) {
      // the legacy default stream cannot be captured into a graph: use an own *blocking* stream, which keeps the
      // implicit ordering with work the caller enqueues on the default stream
      FR_CUDA_TRY(cudaStreamCreate(&stream));
      own_stream = true;
    }
    FR_REQUIRE(c->gamma > 1.0, "gamma must be > 1");
    const bool ns = system == FR_NAVIER_STOKES;
    FR_REQUIRE(!ns || (c->mu >= 0.0 && c->prandtl > 0.0), "mu must be >= 0 and prandtl > 0");
    FR_REQUIRE(!ns || (std::isfinite(c->ldg_beta) && std::isfinite(c->ldg_tau)), "ldg_beta and ldg_tau must be finite");
    FR_REQUIRE(std::isfinite(c->gamma) && (!ns || (std::isfinite(c->mu) && std::isfinite(c->prandtl))), "gamma, mu and prandtl must be finite");
    ph.gamma = (T)c->gamma;
    ph.mu = (T)(ns ? c->mu : 0.0);
    ph.prandtl = (T)(ns ? c->prandtl : 1.0);
    ph.beta = (T)(ns ? c->ldg_beta : 0.0);
    ph.tau = (T)(ns ? c->ldg_tau : 0.0);
    ph.ns = ns ? 1 : 0;
    nt = c->netypes;
    FR_REQUIRE(nt >= 1 && nt <= FR_MAXTYPES && c->eles, "netypes must be in [1,4] and eles non-NULL");
    FR_REQUIRE(c->ifaces, "ifaces must be non-NULL");

    long long utot = 0, gtot = 0;
    for (int t = 0; t < nt; ++t) {
      const fr_eles_desc &d = c->eles[t];
      FR_REQUIRE(d.etype == FR_TET || d.etype == FR_PRI || d.etype == FR_HEX, "unknown element type");
      FR_REQUIRE(d.order >= 1 && d.nupts > 0 && d.nfpts > 0 && d.nfpts < 65536 && d.neles > 0 &&
                     d.neles < (1ll << 31) - 128,
                 "bad element counts");
      const int p = d.order;
      const int nu = d.etype == FR_TET ? (p + 1) * (p + 2) * (p + 3) / 6
                     : d.etype == FR_PRI ? (p + 1) * (p + 1) * (p + 2) / 2 : (p + 1) * (p + 1) * (p + 1);
      const int nf = d.etype == FR_TET ? 2 * (p + 1) * (p + 2)
                     : d.etype == FR_PRI ? (p + 1) * (p + 2) + 3 * (p + 1) * (p + 1) : 6 * (p + 1) * (p + 1);
      FR_REQUIRE(nu == d.nupts && nf == d.nfpts, "nupts / nfpts do not match the element type and order (Table 2)");
      FR_REQUIRE(d.M0 && d.M132 && d.M3 && d.smats && d.rcpdjac, "operator / metric pointers must be non-NULL");
      FR_REQUIRE(!ns || (d.M460 && d.M6), "M460 and M6 are required for Navier-Stokes");
      auto e = std::make_unique<EleData<T>>();
      tname[t] = d.etype == FR_TET ? "tet" : (d.etype == FR_PRI ? "pri" : "hex");
      EleView<T> &v = e->view;
      v.nupts = nu;
      v.nfpts = nf;
      v.affine = d.affine ? 1 : 0;
      v.neles = d.neles;
      v.ld = (d.neles + 127) / 128 * 128;   // whole panels of up to 128 elements (panel.cuh)
      const long long ld = v.ld, ne = d.neles;
      // metric terms, padded with the identity so padding lanes stay finite
      const long long npt = v.affine ? 1 : nu;
      std::vector<T> sm((size_t)9 * npt * ld, T(0)), rj((size_t)npt * ld, T(1));
      for (int ai = 0; ai < 9; ++ai)
        for (long long r = 0; r < npt; ++r) {
          const double *src = d.smats + ((size_t)ai * npt + r) * ne;
          T *dst = sm.data() + ((size_t)ai * npt + r) * ld;
          for (long long k = 0; k < ne; ++k) dst[k] = (T)src[k];
          if (ai % 4 == 0)
            for (long long k = ne; k < ld; ++k) dst[k] = T(1);
        }
      for (long long r = 0; r < npt; ++r)
        for (long long k = 0; k < ne; ++k) {
          const double x = d.rcpdjac[(size_t)r * ne + k];
          FR_REQUIRE(x > 0.0 && std::isfinite(x), "rcpdjac must be positive and finite");
          rj[(size_t)r * ld + k] = (T)x;
        }
      e->smats.upload(sm);
      e->rcpdjac.upload(rj);
      v.smats = e->smats.p;
      v.rcpdjac = e->rcpdjac.p;
      gemm_plan_build(e->pM0, nf, nu, d.M0);
      gemm_plan_build(e->pM132, nu, 3 * nu, d.M132);
      gemm_plan_build(e->pM3, nu, nf, d.M3);
      if (ns) {
        gemm_plan_build(e->pM460, 3 * nu, nu, d.M460);
        gemm_plan_build(e->pM6, 3 * nu, nf, d.M6);
      }
      if (mode == FR_MODE_FUSED) {
        build_split(e->pDiv, nu, [&](PanelOp<T> &op, int r0, int nr) { return fused_div_build(op, nu, nf, d.M132, d.M3, 0, r0, nr); });
        if (ns)
          build_split(e->pGrad, nu,
                      [&](PanelOp<T> &op, int r0, int nr) { return fused_grad_build(op, nu, nf, d.M460, d.M6, 0, d.M0, r0, nr); });
      }
      const size_t nstate = (size_t)nu * 5 * ld;
      e->X.alloc(nstate);
      e->Y.alloc(nstate);
      if (stepper == FR_RK4) e->ACC.alloc(nstate);
      e->grad.alloc(3 * nstate);
      e->R.alloc(nstate);
      tt.ubase[t] = utot;
      tt.gbase[t] = gtot;
      tt.ld[t] = ld;
      tt.gcomp[t] = (long long)nf * 5 * ld;
      utot += (long long)nf * 5 * ld;
      gtot += 3ll * nf * 5 * ld;
      el.push_back(std::move(e));
    }
    for (int t = nt; t < FR_MAXTYPES; ++t) tt.ubase[t] = tt.gbase[t] = tt.ld[t] = tt.gcomp[t] = 0;
    if (c->halo && c->halo->nghost > 0) {
      FR_REQUIRE(nt < FR_MAXTYPES, "a halo needs a free element-type slot (at most 3 element types per rank)");
      FR_REQUIRE(c->halo->et && c->halo->fpt && c->halo->ele, "halo arrays must be non-NULL");
      nghost = c->halo->nghost;
      const long long ldg = (nghost + 127) / 128 * 128;
      tt.ubase[nt] = utot;
      tt.gbase[nt] = gtot;
      tt.ld[nt] = ldg;
      tt.gcomp[nt] = 5 * ldg;                 // one flux point per ghost "element"
      utot += 5 * ldg;
      gtot += 15 * ldg;
    }
    if (mode == FR_MODE_FUSED && ns) {
      // the jump formulation of S2 needs every type on the fused gradient kernel; otherwise fall back to C itself
      bool all = true;
      for (int t = 0; t < nt; ++t) all = all && !el[t]->pGrad.empty();
      if (all) {
        jump = 1;
      } else {
        for (int t = 0; t < nt; ++t)
          if (!el[t]->pGrad.empty()) {
            const fr_eles_desc &d = c->eles[t];
            build_split(el[t]->pGrad, d.nupts, [&](PanelOp<T> &op, int r0, int nr) {
              return fused_grad_build(op, d.nupts, d.nfpts, d.M460, d.M6, 0, nullptr, r0, nr);
            });
          }
      }
    }
    uf.alloc(utot);
    if (ns) {
      cf.alloc(utot);
      gf.alloc(gtot);
    }
    build_views(c);
    if (mode == FR_MODE_FUSED) autotune(c);
    coef.alloc(8);
    FR_CUDA_TRY(cudaMallocHost(&coef_host, 8 * sizeof(StageCoef)));
    for (int i = 0; i < 8; ++i) coef_host[i] = StageCoef{0.0, 0.0};
    FR_CUDA_TRY(cudaDeviceSynchronize());
  }

  // ------------------------------------------------------------------ geometry autotuning
  // The static score of choose_geom ranks the (warps x row groups x column blocks x warp groups) candidates of an operator;
  // which one is fastest depends on things it does not model (register allocation, barrier skew, epilogue latency).  For
  // meshes large enough to time reliably, fr_setup launches the first kTuneCands candidates on the context's own arrays and
  // keeps the fastest.  Results do not depend on the choice: bit-identical for every geometry (tests/test_gpu_parity.py).
  static constexpr int kTuneCands = 14;
  static constexpr long long kTuneMinEles = 16384;
  template <typename B, typename L>
  void tune(PanelOp<T> &cur, B build, L launch, const char *what) {
    if (!cur.ok()) return;
    cudaEvent_t e0, e1;
    FR_CUDA_TRY(cudaEventCreate(&e0));
    FR_CUDA_TRY(cudaEventCreate(&e1));
    // minimum of three single launches after a warm-up: a mean of two was seen 56 % off for one candidate in one of two otherwise
    // identical runs (profiles/r01_j_panel_source_level.md), enough to mis-rank geometries
    auto time_op = [&](const PanelOp<T> &op) {
      launch(op);
      float best_ms = 1e30f;
      for (int rep = 0; rep < 3; ++rep) {
        cudaEventRecord(e0, stream);
        launch(op);
        cudaEventRecord(e1, stream);
        FR_CUDA_TRY(cudaEventSynchronize(e1));
        float ms = 0;
        cudaEventElapsedTime(&ms, e0, e1);
        best_ms = std::min(best_ms, ms);
      }
      return best_ms;
    };
    PanelOp<T> best = cur;
    float bt = time_op(best);
#ifdef FRB_DEBUG_KNOBS
    const bool verbose = getenv("FRB_PANEL_VERBOSE") != nullptr;
#else
    const bool verbose = false;
#endif
    if (verbose) fprintf(stderr, "autotune %s cand 0: %.3f ms\n", what, bt);
    // only the launch geometry varies between candidates: the packing (k-lists or dense k-blocks) and the composition of every
    // k-block depend on the operator alone (panel.cuh), so every candidate gives bit-identical results
    const int ncand = getenv("FRB_TUNE_CANDS") ? std::max(1, atoi(getenv("FRB_TUNE_CANDS"))) : kTuneCands;
    for (int k = 1; k < ncand; ++k) {
      PanelOp<T> op;
      if (!build(op, k)) break;   // candidates are the geometries that fit shared memory, in order: no k-th one left
      const float t = time_op(op);
      if (verbose) fprintf(stderr, "autotune %s cand %d: %.3f ms\n", what, k, t);
      if (t < bt) {
        panel_op_free(best);
        best = op;
        bt = t;
      } else {
        panel_op_free(op);
      }
    }
    cur = best;
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
  }

  void autotune(const fr_config *c) {
    const char *env = getenv("FRB_AUTOTUNE");
    if (env && atoi(env) == 0) return;
    const bool ns = ph.ns;
    for (int t = 0; t < nt; ++t) {
      EleData<T> &e = *el[t];
      if (e.view.neles < kTuneMinEles) continue;
      const fr_eles_desc &d = c->eles[t];
      const int nu = e.view.nupts, nf = e.view.nfpts;
      const long long n5 = 5 * e.view.ld;
      T *ufp = uf.p + tt.ubase[t];
      std::string tag = std::string(tname[t]);
      if (e.pM0.pop)
        tune(*e.pM0.pop, [&](PanelOp<T> &op, int k) { return panel_gemm_build(op, nf, nu, d.M0, k); },
             [&](const PanelOp<T> &op) {
               // both uses of M0: S1, and (Navier-Stokes) S5 on the three gradient components, which is three quarters of its time
               panel_gemm_run(op, n5, T(1), (const T *)e.X.p, n5, 0, T(0), ufp, n5, 0, 1, stream);
               if (ns) panel_gemm_run(op, n5, T(1), (const T *)e.grad.p, n5, (long long)nu * n5, T(0), gf.p + tt.gbase[t], n5, tt.gcomp[t], 3, stream);
             },
             (tag + ":M0").c_str());
      StageArgs<T> plain{nullptr, nullptr, nullptr, e.R.p, nullptr};
      for (auto &q : e.pDiv)
        tune(q.op, [&](PanelOp<T> &op, int k) { return fused_div_build(op, nu, nf, d.M132, d.M3, k, q.r0, q.nr); },
             [&](const PanelOp<T> &op) { launch_fused_div(op, e.view, (const T *)e.grad.p, (const T *)ufp, plain, stream); },
             (tag + ":[M132|M3]").c_str());
      if (ns)
        for (auto &q : e.pGrad)
          tune(q.op,
               [&](PanelOp<T> &op, int k) { return fused_grad_build(op, nu, nf, d.M460, d.M6, k, jump ? d.M0 : nullptr, q.r0, q.nr); },
               [&](const PanelOp<T> &op) {
                 launch_fused_grad(op, e.view, (const T *)e.X.p, (const T *)(cf.p + tt.ubase[t]), e.grad.p, stream);
               },
               (tag + ":[M460|M6]").c_str());
    }
    FR_CUDA_TRY(cudaStreamSynchronize(stream));
  }

  void build_views(const fr_config *c) {
    const fr_iface_desc &f = *c->ifaces;
    FR_REQUIRE(f.npairs >= 0, "npairs must be >= 0");
    FR_REQUIRE(f.npairs == 0 || (f.l_et && f.l_fpt && f.l_ele && f.r_et && f.r_fpt && f.r_ele && f.nl && f.magl && f.magr),
               "interface arrays must be non-NULL");
    // every (type, element, flux point) exactly once across pairs and boundaries
    std::vector<std::vector<uint8_t>> seen(nt);
    for (int t = 0; t < nt; ++t) seen[t].assign(((size_t)el[t]->view.nfpts * el[t]->view.neles + 7) / 8, 0);
    std::vector<uint8_t> gseen((size_t)nghost, 0);
    auto visit = [&](int t, long long e, int s) {
      if (t == nt && nghost > 0) {           // the remote side of a cut pair
        FR_REQUIRE(s == 0 && e >= 0 && e < nghost, "ghost reference out of range");
        FR_REQUIRE(!gseen[(size_t)e], "a ghost is referenced more than once");
        gseen[(size_t)e] = 1;
        return;
      }
      FR_REQUIRE(t >= 0 && t < nt, "flux-point reference: element type out of range");
      FR_REQUIRE(e >= 0 && e < el[t]->view.neles && s >= 0 && s < el[t]->view.nfpts,
                 "flux-point reference: element or flux point out of range");
      const size_t bit = (size_t)s * el[t]->view.neles + e;
      FR_REQUIRE(!(seen[t][bit >> 3] & (1u << (bit & 7))), "a flux point is referenced more than once");
      seen[t][bit >> 3] |= (uint8_t)(1u << (bit & 7));
    };
    const long long np = f.npairs;
    for (long long k = 0; k < np; ++k) {
      visit(f.l_et[k], f.l_ele[k], f.l_fpt[k]);
      visit(f.r_et[k], f.r_ele[k], f.r_fpt[k]);
    }
    FR_REQUIRE(c->nbcs >= 0 && (c->nbcs == 0 || c->bcs), "bcs must be non-NULL when nbcs > 0");
    for (int b = 0; b < c->nbcs; ++b) {
      const fr_bc_desc &d = c->bcs[b];
      FR_REQUIRE(d.type == FR_BC_NOSLIP_ISOTHERMAL_WALL || d.type == FR_BC_CHAR_RIEMANN_INV, "unknown boundary type");
      FR_REQUIRE(d.nfpts >= 0 && (d.nfpts == 0 || (d.et && d.fpt && d.ele && d.n && d.mag)), "boundary arrays must be non-NULL");
      for (long long k = 0; k < d.nfpts; ++k) visit(d.et[k], d.ele[k], d.fpt[k]);
    }
    for (int t = 0; t < nt; ++t) {
      const size_t nbits = (size_t)el[t]->view.nfpts * el[t]->view.neles;
      size_t cnt = 0;
      for (uint8_t b : seen[t]) cnt += __builtin_popcount(b);
      FR_REQUIRE(cnt == nbits, "unpaired flux points: every flux point must appear in a pair or a boundary list");
    }
    for (long long g = 0; g < nghost; ++g) FR_REQUIRE(gseen[(size_t)g], "every ghost must be the remote side of exactly one pair");
    if (nghost > 0) {
      // the own side of every cut pair: where its U_f and G_f sit in the flat arrays
      const fr_halo_desc &h = *c->halo;
      std::vector<long long> ou(nghost), og(nghost), hl(nghost), hg(nghost), ps(nghost, 0), pc(nghost, nghost), pj(nghost);
      for (long long g = 0; g < nghost; ++g) {
        const int t = h.et[g];
        FR_REQUIRE(t >= 0 && t < nt && h.ele[g] >= 0 && h.ele[g] < el[t]->view.neles && h.fpt[g] >= 0 && h.fpt[g] < el[t]->view.nfpts,
                   "halo send entry out of range");
        const size_t bit = (size_t)h.fpt[g] * el[t]->view.neles + h.ele[g];
        FR_REQUIRE(seen[t][bit >> 3] & (1u << (bit & 7)), "halo send entry is not a flux point of this rank");
        const long long rel = (long long)h.fpt[g] * 5 * tt.ld[t] + h.ele[g];
        ou[g] = tt.ubase[t] + rel;
        og[g] = tt.gbase[t] + rel;
        hl[g] = tt.ld[t];
        hg[g] = tt.gcomp[t];
        pj[g] = g;
      }
      h_offu.upload(ou);
      h_offg.upload(og);
      h_ld.upload(hl);
      h_gcomp.upload(hg);
      h_pstart.upload(ps);
      h_pcnt.upload(pc);
      h_pj.upload(pj);
      hv = HaloView{nghost, h_offu.p, h_offg.p, h_ld.p, h_gcomp.p, h_pstart.p, h_pcnt.p, h_pj.p,
                    tt.ubase[nt], tt.gbase[nt], tt.ld[nt], tt.gcomp[nt]};
      h_send[0].alloc((size_t)5 * nghost);
      h_recv[0].alloc((size_t)5 * nghost);
      if (ph.ns) {
        h_send[1].alloc((size_t)15 * nghost);
        h_recv[1].alloc((size_t)15 * nghost);
      }
    }
    // Pairs sorted by (type_L, block of kIfaceBlock consecutive e_L, sigma_L, e_L): inside a block the L side is read and written
    // in coalesced runs, and all flux points of a neighbourhood of elements are visited within a short time window, so the 32-byte
    // sectors of the scattered R side (8 useful bytes per access) are completed out of L1/L2 instead of being fetched from DRAM
    // once per access (a plain (type, sigma, e) order moved 2.2x / 1.6x the algorithmic bytes in S2 / S7, profiles/r01_d_launches.md).
    const long long blk = getenv("FRB_IFACE_BLOCK") ? atoll(getenv("FRB_IFACE_BLOCK")) : kIfaceBlock;
    std::vector<long long> order(np);
    std::iota(order.begin(), order.end(), 0ll);
    auto key_less = [&](long long a, long long b) {
      if (f.l_et[a] != f.l_et[b]) return f.l_et[a] < f.l_et[b];
      const long long ba = f.l_ele[a] / blk, bb = f.l_ele[b] / blk;
      if (ba != bb) return ba < bb;
      if (f.l_fpt[a] != f.l_fpt[b]) return f.l_fpt[a] < f.l_fpt[b];
      return f.l_ele[a] < f.l_ele[b];
    };
    if (!std::is_sorted(order.begin(), order.end(), key_less)) std::sort(order.begin(), order.end(), key_less);
    std::vector<PairRec> pr(np);
    std::vector<T> hn(3 * (size_t)np), hl(np), hr(np);
    for (long long i = 0; i < np; ++i) {
      const long long k = order[i];
      pr[i] = PairRec{(int)f.l_ele[k], (f.l_et[k] << 16) | f.l_fpt[k], (int)f.r_ele[k], (f.r_et[k] << 16) | f.r_fpt[k]};
      double nn = 0;
      for (int d = 0; d < 3; ++d) {
        hn[(size_t)d * np + i] = (T)f.nl[(size_t)d * np + k];
        nn += f.nl[(size_t)d * np + k] * f.nl[(size_t)d * np + k];
      }
      FR_REQUIRE(std::fabs(nn - 1.0) < 1e-6, "interface normals must be unit vectors");
      FR_REQUIRE(f.magl[k] > 0 && f.magr[k] > 0, "interface magnitudes must be positive");
      hl[i] = (T)f.magl[k];
      hr[i] = (T)f.magr[k];
    }
    pairs.upload(pr);
    nl.upload(hn);
    magl.upload(hl);
    magr.upload(hr);
    iv.npairs = np;
    iv.pairs = pairs.p;
    iv.nl = nl.p;
    iv.magl = magl.p;
    iv.magr = magr.p;
    for (int b = 0; b < c->nbcs; ++b) {
      const fr_bc_desc &d = c->bcs[b];
      auto bd = std::make_unique<BndData<T>>();
      const long long n = d.nfpts;
      std::vector<BndRec> rec(n);
      std::vector<T> bn(3 * (size_t)n), bm(n);
      for (long long k = 0; k < n; ++k) {
        rec[k] = BndRec{(int)d.ele[k], (d.et[k] << 16) | d.fpt[k]};
        for (int q = 0; q < 3; ++q) bn[(size_t)q * n + k] = (T)d.n[(size_t)q * n + k];
        bm[k] = (T)d.mag[k];
      }
      bd->recs.upload(rec);
      bd->nrm.upload(bn);
      bd->mag.upload(bm);
      bd->view.n = n;
      bd->view.type = (int)d.type;
      bd->view.recs = bd->recs.p;
      bd->view.nrm = bd->nrm.p;
      bd->view.mag = bd->mag.p;
      for (int q = 0; q < 8; ++q) bd->view.par[q] = (T)d.params[q];
      bnd.push_back(std::move(bd));
    }
  }

  // ------------------------------------------------------------------ one RHS evaluation (S1..S9/S10)
  // u[t]: stage input; sa[t]: what the last kernel of type t writes.  Returns kernels launched.
  // mask: which of the three phases between the halo exchanges run (include/frb200.h fr_rhs_phase); 7 = the whole right-hand side.
  // With a halo, a whole evaluation in one call is only meaningful when the caller has filled the receive buffers some other way.
  int run_rhs(const T *const *u, const StageArgs<T> *sa, Timeline *tl, int mask = 7) {
    int nk = 0;
    cudaStream_t s = stream;
    const bool ns = ph.ns;
    const double w = sizeof(T);
    auto mark = [&](int c, int t, const char *step, double words, double fl) {
      if (!tl) return;
      std::string nm = t >= 0 ? std::string(tname[t]) + ":" + step : std::string(step);
      tl->mark(c, nm, words * w, fl);
    };
    if (tl) tl->mark(-1);
    double nbnd = 0;
    for (auto &b : bnd) nbnd += (double)b->view.n;
    const double npr = (double)iv.npairs;
    auto do_S1 = [&](int t, cudaStream_t q) {   // S1: U_f = M0 U
      NvtxRange r("S1 interp");
      EleData<T> &e = *el[t];
      const double n = (double)e.view.neles, nu = e.view.nupts, nf = e.view.nfpts;
      nk += gemm_run(e.pM0, 5 * e.view.ld, T(1), u[t], 5 * e.view.ld, 0, T(0), uf.p + tt.ubase[t], 5 * e.view.ld, 0, 1, q);
      mark(CAT_GEMM, t, "S1_M0", (nu + nf) * 5 * n, 2 * (e.pM0.pop ? e.pM0.pop->density : 1.0) * nf * nu * 5 * n);
    };
    auto do_S2 = [&]() {
      NvtxRange r("S2 con_u");
      nk += launch_con_u(iv, tt, uf.p, cf.p, ph.beta, jump, s);   // S2
      for (auto &b : bnd) nk += launch_bc_con_u(b->view, tt, uf.p, cf.p, ph.gamma, jump, s);
      const double words = jump ? (ph.beta == T(0.5) ? 15 : 20) : 20;
      mark(CAT_IFACE, -1, jump ? "S2_con_u_jump" : "S2_con_u", npr * (words + 16 / w) + nbnd * (10 + 3 + 8 / w), npr * 15 + nbnd * 60);
    };
    auto do_grad = [&](int t, cudaStream_t q) {   // S3, S4, S5
      NvtxRange r("S3-S5 gradient");
      EleData<T> &e = *el[t];
      const long long n5 = 5 * e.view.ld;
      const double n = (double)e.view.neles, nu = e.view.nupts, nf = e.view.nfpts;
      const double nmet = e.view.affine ? 1 : nu;
      if (!e.pGrad.empty()) {
        // S3 + S4 fused: G = (1/|J|) S^T ([M460 | M6] [U; C])
        for (auto &g : e.pGrad) nk += launch_fused_grad(g.op, e.view, u[t], cf.p + tt.ubase[t], e.grad.p, q);
        mark(CAT_GEMM, t, "S3_S4_fused_grad", (5 * nu + 5 * nf + 15 * nu + 10 * nmet) * n,
             2 * parts_density(e.pGrad) * 3 * nu * (nu + nf) * 5 * n + 15 * 6 * nu * n);
      } else {
        // S3: G~ = M460 U + M6 C
        nk += gemm_run(e.pM460, n5, T(1), u[t], n5, 0, T(0), e.grad.p, n5, 0, 1, q);
        mark(CAT_GEMM, t, "S3a_M460", (nu + 3 * nu) * 5 * n, 2 * 3 * nu * nu * 5 * n);
        nk += gemm_run(e.pM6, n5, T(1), cf.p + tt.ubase[t], n5, 0, T(1), e.grad.p, n5, 0, 1, q);
        mark(CAT_GEMM, t, "S3b_M6", (nf + 6 * nu) * 5 * n, 2 * 3 * nu * nf * 5 * n);
        nk += launch_gradcoru(e.view, e.grad.p, q);   // S4
        mark(CAT_PW, t, "S4_gradcoru", (30 * nu + 10 * nmet) * n, 15 * 6 * nu * n);
      }
      // S5: G_f,i = M0 G_i, i = 0..2 (batched)
      nk += gemm_run(e.pM0, n5, T(1), e.grad.p, n5, (long long)e.view.nupts * n5, T(0), gf.p + tt.gbase[t], n5,
                     tt.gcomp[t], 3, q);
      mark(CAT_GEMM, t, "S5_M0grad", (nu + nf) * 15 * n, 2 * (e.pM0.pop ? e.pM0.pop->density : 1.0) * nf * nu * 15 * n);
    };
    auto do_S7 = [&]() {
      NvtxRange r("S7 comm_flux");
      nk += launch_comm_flux(iv, tt, uf.p, gf.p, ph, s);   // S7 (D overwrites U_f)
      for (auto &b : bnd) nk += launch_bc_comm_flux(b->view, tt, uf.p, gf.p, ph, s);
      const double sides = ns ? ((ph.beta == T(0.5) || ph.beta == T(-0.5)) ? 1 : 2) : 0;
      mark(CAT_IFACE, -1, "S7_comm_flux", npr * (20 + 15 * sides + 5 + 16 / w) + nbnd * (10 + (ns ? 15 : 0) + 4 + 8 / w),
           npr * (ns ? 420 : 160) + nbnd * (ns ? 420 : 200));
    };
    auto do_S6 = [&](int t, cudaStream_t q) {
      NvtxRange r("S6 tdisf");
      EleData<T> &e = *el[t];
      const double n = (double)e.view.neles, nu = e.view.nupts;
      const double nmet = e.view.affine ? 1 : nu;
      nk += launch_tdisf(e.view, u[t], e.grad.p, ph, q);   // S6 (Euler, or unfused): F~ in place over G
      mark(CAT_PW, t, "S6_tdisf", ((ns ? 35 : 20) * nu + 9 * nmet) * n, (ns ? 210 : 110) * nu * n);
    };
    auto do_div = [&](int t, cudaStream_t q) {   // S8, S9, S10
      NvtxRange r("S8-S10 divergence + stage update");
      EleData<T> &e = *el[t];
      const long long n5 = 5 * e.view.ld;
      const double n = (double)e.view.neles, nu = e.view.nupts, nf = e.view.nfpts;
      const double nmet = e.view.affine ? 1 : nu;
      const T *ft = e.grad.p;
      if (!e.pDiv.empty()) {
        // S8 + S9 (+S10) fused: out = -(1/|J|) [M132 | M3] [F~; D], stage update in the epilogue
        for (auto &g : e.pDiv) nk += launch_fused_div(g.op, e.view, ft, uf.p + tt.ubase[t], sa[t], q);
        const double rk = sa[t].coef ? (sa[t].out2 ? 15 : 10) : 5;
        mark(CAT_GEMM, t, sa[t].coef ? "S8_S9_S10_fused_div_rk" : "S8_S9_fused_div", (15 * nu + 5 * nf + rk * nu + nmet) * n,
             2 * parts_density(e.pDiv) * nu * (3 * nu + nf) * 5 * n + 5 * nu * n);
        return;
      }
      // S8: R = M132 F~ + M3 D
      nk += gemm_run(e.pM132, n5, T(1), e.grad.p, n5, 0, T(0), e.R.p, n5, 0, 1, q);
      mark(CAT_GEMM, t, "S8a_M132", (3 * nu + nu) * 5 * n, 2 * nu * 3 * nu * 5 * n);
      nk += gemm_run(e.pM3, n5, T(1), uf.p + tt.ubase[t], n5, 0, T(1), e.R.p, n5, 0, 1, q);
      mark(CAT_GEMM, t, "S8b_M3", (nf + 2 * nu) * 5 * n, 2 * nu * nf * 5 * n);
      nk += launch_negdivconf(e.view, e.R.p, sa[t], q);   // S9 / S10
      const double extra = sa[t].coef ? (sa[t].out2 ? 20 : 10) : 5;
      mark(CAT_PW, t, sa[t].coef ? "S9_S10_negdiv_rk" : "S9_negdivconf", ((5 + extra) * nu + nmet) * n, 5 * nu * n * (sa[t].coef ? 5 : 1));
    };
    if (!tl && cmask && nt > 1 && mask == 7 && !nghost) {
      // The element types' chains are independent between the interface kernels (which read and write every type's flux
      // points): a phase whose bit is set in cmask runs one branch per type (1: S1, 2: S3..S5, 4: S6 beside S7, 8: S8..S10),
      // the interface kernels stay on the caller's stream.  Under capture the events become the edges of the step's graph.
      ensure_branches();
      auto rec = [&](cudaEvent_t e, cudaStream_t q) { FR_CUDA_TRY(cudaEventRecord(e, q)); };
      auto wait = [&](cudaStream_t q, cudaEvent_t e) { FR_CUDA_TRY(cudaStreamWaitEvent(q, e, 0)); };
      auto branch = [&](int t, int bit) { return (cmask & bit) ? aux[t] : s; };
      auto fork_join = [&](int bit, cudaEvent_t start, auto &&body) {
        if (cmask & bit) rec(start, s);
        for (int t = 0; t < nt; ++t) {
          cudaStream_t q = branch(t, bit);
          if (q != s) wait(q, start);
          body(t, q);
          if (q != s) rec(ev_type[t], q);
        }
        if (cmask & bit)
          for (int t = 0; t < nt; ++t) wait(s, ev_type[t]);
      };
      fork_join(1, ev_main[0], do_S1);
      if (ns) {
        do_S2();
        fork_join(2, ev_main[1], do_grad);
      }
      if (cmask & 4) {                       // S6 needs only this evaluation's S5 to have read G: beside S7
        rec(ev_main[1], s);
        for (int t = 0; t < nt; ++t) {
          wait(aux[t], ev_main[1]);
          do_S6(t, aux[t]);
          rec(ev_type[t], aux[t]);
        }
      }
      do_S7();
      if (!(cmask & 4))
        for (int t = 0; t < nt; ++t) do_S6(t, s);
      if (cmask & 8) rec(ev_main[2], s);
      for (int t = 0; t < nt; ++t) {
        cudaStream_t q = branch(t, 8);
        if (q != s) wait(q, ev_main[2]);     // S7 (and S6 where it ran on s); S6 on aux[t] precedes in stream order
        else if (cmask & 4) wait(s, ev_type[t]);
        do_div(t, q);
        if (q != s) rec(ev_type[t], q);
      }
      if (cmask & 8)
        for (int t = 0; t < nt; ++t) wait(s, ev_type[t]);
      return nk;
    }
    if (mask & 1) {
      for (int t = 0; t < nt; ++t) do_S1(t, s);
      if (nghost) nk += launch_halo_pack(hv, 0, (const T *)uf.p, h_send[0].p, s);
    }
    if (mask & 2) {
      if (nghost) nk += launch_halo_unpack(hv, 0, (const T *)h_recv[0].p, uf.p, s);
      if (ns) {
        do_S2();
        for (int t = 0; t < nt; ++t) do_grad(t, s);
        if (nghost) nk += launch_halo_pack(hv, 1, (const T *)gf.p, h_send[1].p, s);
      }
    }
    if (mask & 4) {
      if (nghost && ns) nk += launch_halo_unpack(hv, 1, (const T *)h_recv[1].p, gf.p, s);
      do_S7();
      for (int t = 0; t < nt; ++t) {
        do_S6(t, s);
        do_div(t, s);
      }
    }
    return nk;
  }

  // per-type branch streams and the events that fork from / join into the caller's stream (run_rhs)
  void ensure_branches() {
    if ((int)aux.size() == nt) return;
    for (int t = (int)aux.size(); t < nt; ++t) {
      cudaStream_t q;
      cudaEvent_t e;
      FR_CUDA_TRY(cudaStreamCreateWithFlags(&q, cudaStreamNonBlocking));
      aux.push_back(q);
      FR_CUDA_TRY(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
      ev_type.push_back(e);
    }
    for (int i = 0; i < 3; ++i)
      if (!ev_main[i]) FR_CUDA_TRY(cudaEventCreateWithFlags(&ev_main[i], cudaEventDisableTiming));
  }

  void state_layout(int et, int64_t *ld, int64_t *nbytes) const override {
    FR_REQUIRE(et >= 0 && et < nt, "element type index out of range");
    if (ld) *ld = el[et]->view.ld;
    if (nbytes) *nbytes = (int64_t)el[et]->view.nupts * 5 * el[et]->view.ld * (int64_t)sizeof(T);
  }

  void rhs(const void *const *u, void *const *dudt) override {
    FR_REQUIRE(u && dudt, "u_dev and dudt_dev must be non-NULL");
    std::vector<const T *> up(nt);
    std::vector<StageArgs<T>> sa(nt);
    for (int t = 0; t < nt; ++t) {
      FR_REQUIRE(u[t] && dudt[t] && u[t] != dudt[t], "state pointers must be non-NULL and must not alias");
      FR_REQUIRE(((uintptr_t)u[t] % 16) == 0 && ((uintptr_t)dudt[t] % 16) == 0, "state pointers must be 16-byte aligned");
      up[t] = (const T *)u[t];
      sa[t] = StageArgs<T>{nullptr, nullptr, nullptr, (T *)dudt[t], nullptr};
    }
    launches += run_rhs(up.data(), sa.data(), nullptr);
  }

  void set_state(const double *const *u) override {
    FR_REQUIRE(u, "u_host must be non-NULL");
    for (int t = 0; t < nt; ++t) {
      FR_REQUIRE(u[t], "u_host[t] must be non-NULL");
      const EleView<T> &v = el[t]->view;
      std::vector<T> h((size_t)v.nupts * 5 * v.ld, T(0));
      for (long long r = 0; r < (long long)v.nupts * 5; ++r)
        for (long long k = 0; k < v.neles; ++k) h[(size_t)r * v.ld + k] = (T)u[t][(size_t)r * v.neles + k];
      FR_CUDA_TRY(cudaStreamSynchronize(stream));
      FR_CUDA_TRY(cudaMemcpy(el[t]->X.p, h.data(), h.size() * sizeof(T), cudaMemcpyHostToDevice));
    }
  }

  void get_state(double *const *u) override {
    FR_REQUIRE(u, "u_host must be non-NULL");
    FR_CUDA_TRY(cudaStreamSynchronize(stream));
    for (int t = 0; t < nt; ++t) {
      FR_REQUIRE(u[t], "u_host[t] must be non-NULL");
      const EleView<T> &v = el[t]->view;
      std::vector<T> h((size_t)v.nupts * 5 * v.ld);
      FR_CUDA_TRY(cudaMemcpy(h.data(), el[t]->X.p, h.size() * sizeof(T), cudaMemcpyDeviceToHost));
      for (long long r = 0; r < (long long)v.nupts * 5; ++r)
        for (long long k = 0; k < v.neles; ++k) u[t][(size_t)r * v.neles + k] = (double)h[(size_t)r * v.ld + k];
    }
  }

  // ------------------------------------------------------------------ Runge-Kutta (S10 fused into S9)
  int nstages() const { return stepper == FR_RK4 ? 4 : (stepper == FR_EULER1 ? 1 : 5); }

  void fill_coefs(double dt) {
    if (stepper == FR_RK4) {
      const StageCoef c[4] = {{dt / 6, dt / 2}, {dt / 3, dt / 2}, {dt / 3, dt}, {dt / 6, 0.0}};
      for (int i = 0; i < 4; ++i) coef_host[i] = c[i];
    } else if (stepper == FR_EULER1) {
      coef_host[0] = StageCoef{dt, 0.0};              // forward Euler: X <- X + dt K
    } else {
      // RK4(3)5[2R+]C (reading R12): X += dt b_i K ; Y = X_old + dt a_i K
      for (int i = 0; i < 5; ++i) coef_host[i] = StageCoef{dt * kB45[i], dt * kA45[i]};
    }
  }

  // RK4(3)5[2R+]C (reading R12)
  static constexpr double kA45[5] = {970286171893.0 / 4311952581923.0, 6584761158862.0 / 12103376702013.0,
                                     2251764453980.0 / 15575788980749.0, 26877169314380.0 / 34165994151039.0, 0.0};
  static constexpr double kB45[5] = {1153189308089.0 / 22510343858157.0, 1772645290293.0 / 4653164025191.0,
                                     -1672844663538.0 / 4480602732383.0, 2114624349019.0 / 3568978502595.0,
                                     5198255086312.0 / 14908931495163.0};
  static constexpr double kBhat45[5] = {1016888040809.0 / 7410784769900.0, 11231460423587.0 / 58533540763752.0,
                                        -1563879915014.0 / 6823010717585.0, 606302364029.0 / 971179775848.0,
                                        1097981568119.0 / 3980877426909.0};

  // stage input and fused stage update of stage i (S10 of SURVEY 8(a))
  void stage_args(int i, bool adaptive, std::vector<const T *> &up, std::vector<StageArgs<T>> &sa) {
    const int S = nstages();
    for (int t = 0; t < nt; ++t) {
      EleData<T> &e = *el[t];
      up[t] = i == 0 ? e.X.p : e.Y.p;
      const StageCoef *c = coef.p + i;
      if (stepper == FR_RK4) {
        if (i == 0) sa[t] = StageArgs<T>{c, e.X.p, e.X.p, e.ACC.p, e.Y.p};
        else if (i < 3) sa[t] = StageArgs<T>{c, e.ACC.p, e.X.p, e.ACC.p, e.Y.p};
        else sa[t] = StageArgs<T>{c, e.ACC.p, nullptr, e.X.p, nullptr};
      } else if (stepper == FR_EULER1) {
        sa[t] = StageArgs<T>{c, e.X.p, nullptr, e.X.p, nullptr};
      } else {
        // adaptive: the last stage writes Y_5 = X_4 + dt a_5 K_5 = X_4 too, for the error estimate
        sa[t] = StageArgs<T>{c, e.X.p, e.X.p, e.X.p, (i < S - 1 || adaptive) ? e.Y.p : nullptr};
      }
    }
  }

  void rhs_phase(int phase, const void *const *u, void *const *dudt) override {
    FR_REQUIRE(phase >= 0 && phase <= 2, "phase must be 0, 1 or 2");
    FR_REQUIRE(u && (dudt || phase < 2), "u_dev must be non-NULL (and dudt_dev in phase 2)");
    std::vector<const T *> up(nt);
    std::vector<StageArgs<T>> sa(nt);
    for (int t = 0; t < nt; ++t) {
      FR_REQUIRE(u[t] && ((uintptr_t)u[t] % 16) == 0, "state pointers must be non-NULL and 16-byte aligned");
      up[t] = (const T *)u[t];
      T *o = (phase == 2) ? (T *)dudt[t] : nullptr;
      FR_REQUIRE(phase < 2 || (o && (const T *)o != up[t] && ((uintptr_t)o % 16) == 0), "dudt pointers must be non-NULL, aligned and must not alias u");
      sa[t] = StageArgs<T>{nullptr, nullptr, nullptr, o, nullptr};
    }
    launches += run_rhs(up.data(), sa.data(), nullptr, 1 << phase);
  }

  void rk_stage_phase(double dt, int stage, int phase) override {
    FR_REQUIRE(std::isfinite(dt), "dt must be finite");
    FR_REQUIRE(stage >= 0 && stage < nstages() && phase >= 0 && phase <= 2, "stage or phase out of range");
    if (!(dt == coef_dt)) {
      FR_CUDA_TRY(cudaStreamSynchronize(stream));
      fill_coefs(dt);
      FR_CUDA_TRY(cudaMemcpyAsync(coef.p, coef_host, 8 * sizeof(StageCoef), cudaMemcpyHostToDevice, stream));
      coef_dt = dt;
    }
    std::vector<const T *> up(nt);
    std::vector<StageArgs<T>> sa(nt);
    stage_args(stage, false, up, sa);
    launches += run_rhs(up.data(), sa.data(), nullptr, 1 << phase);
  }

  void halo_buffers(int which, void **send, void **recv, int64_t *n) override {
    FR_REQUIRE(which == 0 || which == 1, "which must be 0 (state) or 1 (gradient)");
    if (send) *send = h_send[which].p;
    if (recv) *recv = h_recv[which].p;
    if (n) *n = (int64_t)h_send[which].n;
  }

  void halo_set_peers(int npeers, const int64_t *start, const int64_t *count) override {
    FR_REQUIRE(nghost > 0, "the context has no halo");
    FR_REQUIRE(npeers > 0 && start && count, "peer arrays must be non-NULL");
    std::vector<long long> ps(nghost), pc(nghost), pj(nghost);
    long long next = 0;
    for (int p = 0; p < npeers; ++p) {
      FR_REQUIRE(start[p] == next && count[p] > 0, "peer segments must tile [0, nghost) in order");
      for (long long j = 0; j < count[p]; ++j) {
        ps[next + j] = start[p];
        pc[next + j] = count[p];
        pj[next + j] = j;
      }
      next += count[p];
    }
    FR_REQUIRE(next == nghost, "peer segments must cover every ghost");
    FR_CUDA_TRY(cudaStreamSynchronize(stream));
    FR_CUDA_TRY(cudaMemcpy(h_pstart.p, ps.data(), ps.size() * sizeof(long long), cudaMemcpyHostToDevice));
    FR_CUDA_TRY(cudaMemcpy(h_pcnt.p, pc.data(), pc.size() * sizeof(long long), cudaMemcpyHostToDevice));
    FR_CUDA_TRY(cudaMemcpy(h_pj.p, pj.data(), pj.size() * sizeof(long long), cudaMemcpyHostToDevice));
  }

  int enqueue_step(bool adaptive = false) {
    int nk = 0;
    const int S = nstages();
    std::vector<const T *> up(nt);
    std::vector<StageArgs<T>> sa(nt);
    for (int i = 0; i < S; ++i) {
      stage_args(i, adaptive, up, sa);
      nk += run_rhs(up.data(), sa.data(), nullptr);
      if (adaptive) {
        // dt (b_i - bhat_i) K_i = g_i (Y_i - X_i)  (rk_adapt.cu)
        const double g = (kB45[i] - kBhat45[i]) / (kA45[i] - kB45[i]);
        const int nb = rk_err_blocks();
        for (int t = 0; t < nt; ++t) {
          EleData<T> &e = *el[t];
          const long long n = (long long)e.view.nupts * 5 * e.view.ld;
          if (i < S - 1)
            nk += launch_rk_err_accum(e.E.p, (const T *)e.Y.p, (const T *)e.X.p, g, i == 0, n, stream);
          else
            nk += launch_rk_err_norm((const T *)e.E.p, (const T *)e.Y.p, (const T *)e.X.p, (const T *)e.U0.p, g, err_dev.p + 1, n,
                                     err_partial.p + (size_t)t * nb, stream);
        }
        if (i == S - 1) nk += launch_rk_err_final(err_partial.p, nt * nb, err_dev.p, stream);
      }
    }
    return nk;
  }

  void rk_adaptive(double t0, double t1, double dt0, double atol, double rtol, long long max_attempts, fr_adapt_stats *st,
                   double *dt_hist, double *err_hist, long long hist_cap) override {
    FR_REQUIRE(stepper == FR_RK45_2R, "adaptive stepping needs an FR_RK45_2R context");
    FR_REQUIRE(std::isfinite(t0) && std::isfinite(t1) && t1 >= t0, "need finite t0 <= t1");
    FR_REQUIRE(dt0 > 0 && std::isfinite(dt0), "dt_init must be positive and finite");
    FR_REQUIRE(atol > 0 && rtol >= 0 && std::isfinite(atol) && std::isfinite(rtol), "need atol > 0 and rtol >= 0");
    FR_REQUIRE(max_attempts > 0, "max_attempts must be positive");
    FR_REQUIRE(hist_cap == 0 || (dt_hist && err_hist), "history buffers must be non-NULL when hist_cap > 0");
    const int nb = rk_err_blocks();
    if (!err_host) {
      for (int t = 0; t < nt; ++t) {
        const size_t n = (size_t)el[t]->view.nupts * 5 * el[t]->view.ld;
        if (!el[t]->E.p) el[t]->E.alloc(n);
        if (!el[t]->U0.p) el[t]->U0.alloc(n);
      }
      if (!err_partial.p) err_partial.alloc((size_t)nt * nb);
      if (!err_dev.p) err_dev.alloc(3);
      FR_CUDA_TRY(cudaMallocHost(&err_host, 3 * sizeof(double)));
      // the allocations zero-fill on the legacy stream, which a non-blocking user stream does not wait for
      FR_CUDA_TRY(cudaDeviceSynchronize());
    }
    FR_CUDA_TRY(cudaStreamSynchronize(stream));
    if (tol_set[0] != atol || tol_set[1] != rtol) {
      err_host[1] = atol;
      err_host[2] = rtol;
      FR_CUDA_TRY(cudaMemcpyAsync(err_dev.p + 1, err_host + 1, 2 * sizeof(double), cudaMemcpyHostToDevice, stream));
      tol_set[0] = atol;
      tol_set[1] = rtol;
    }
    if (!graph_adapt) {
      cudaGraph_t g = nullptr;
      FR_CUDA_TRY(cudaStreamBeginCapture(stream, cudaStreamCaptureModeThreadLocal));
      int nk = 0;
      try {
        for (int t = 0; t < nt; ++t) {
          const size_t nbytes = (size_t)el[t]->view.nupts * 5 * el[t]->view.ld * sizeof(T);
          FR_CUDA_TRY(cudaMemcpyAsync(el[t]->U0.p, el[t]->X.p, nbytes, cudaMemcpyDeviceToDevice, stream));
        }
        nk = enqueue_step(true);
        FR_CUDA_TRY(cudaMemcpyAsync(err_host, err_dev.p, sizeof(double), cudaMemcpyDeviceToHost, stream));
      } catch (...) {
        cudaStreamEndCapture(stream, &g);
        if (g) cudaGraphDestroy(g);
        throw;
      }
      FR_CUDA_TRY(cudaStreamEndCapture(stream, &g));
      cudaError_t e = cudaGraphInstantiate(&graph_adapt, g, 0);
      cudaGraphDestroy(g);
      FR_CUDA_TRY(e);
      graph_adapt_kernels = nk;
    }
    double ndof = 0;
    for (int t = 0; t < nt; ++t) ndof += (double)el[t]->view.nupts * 5.0 * (double)el[t]->view.neles;
    // the controller (reading R25), in FP64 on the host
    const double alpha = 0.7 / 4, beta = 0.4 / 4, safety = 0.8, fmin = 0.3, fmax = 2.5;
    double t = t0, dt = dt0, err_prev = 1.0;
    long long nacc = 0, nrej = 0, natt = 0;
    while (t1 - t > 1e-12 * std::fabs(t1 - t0) && natt < max_attempts) {
      const bool last = dt >= t1 - t;
      const double dtt = last ? t1 - t : dt;
      fill_coefs(dtt);
      FR_CUDA_TRY(cudaMemcpyAsync(coef.p, coef_host, 8 * sizeof(StageCoef), cudaMemcpyHostToDevice, stream));
      coef_dt = dtt;
      FR_CUDA_TRY(cudaGraphLaunch(graph_adapt, stream));
      launches += graph_adapt_kernels;
      FR_CUDA_TRY(cudaStreamSynchronize(stream));
      const double err = std::sqrt(err_host[0] / ndof);
      const bool ok = std::isfinite(err) && err <= 1.0;
      if (natt < hist_cap) {
        dt_hist[natt] = dtt;
        err_hist[natt] = err;
      }
      ++natt;
      if (ok) {
        ++nacc;
        t = last ? t1 : t + dtt;
      } else {
        ++nrej;
        for (int tt_ = 0; tt_ < nt; ++tt_) {
          const size_t nbytes = (size_t)el[tt_]->view.nupts * 5 * el[tt_]->view.ld * sizeof(T);
          FR_CUDA_TRY(cudaMemcpyAsync(el[tt_]->X.p, el[tt_]->U0.p, nbytes, cudaMemcpyDeviceToDevice, stream));
        }
      }
      double fac = fmin;
      if (std::isfinite(err)) fac = std::min(fmax, std::max(fmin, safety * std::pow(std::max(err, 1e-10), -alpha) * std::pow(err_prev, beta)));
      dt = dtt * fac;
      if (ok) err_prev = std::max(err, 1e-10);
    }
    FR_CUDA_TRY(cudaStreamSynchronize(stream));
    if (st) {
      st->accepted = nacc;
      st->rejected = nrej;
      st->t = t;
      st->dt_next = dt;
    }
    if (t1 - t > 1e-12 * std::fabs(t1 - t0)) throw Error{FR_ESTATE, "fr_rk_adaptive_run: max_attempts reached before t1"};
  }

  void rk_step(double dt, long long nsteps) override {
    FR_REQUIRE(std::isfinite(dt), "dt must be finite");
    if (nsteps <= 0) return;
    if (!(dt == coef_dt)) {
      FR_CUDA_TRY(cudaStreamSynchronize(stream));   // pinned staging buffer may still be in use
      fill_coefs(dt);
      FR_CUDA_TRY(cudaMemcpyAsync(coef.p, coef_host, 8 * sizeof(StageCoef), cudaMemcpyHostToDevice, stream));
      coef_dt = dt;
    }
    if (!graph) {
      // capture one step; the launchers' cudaFuncSetAttribute calls are not stream operations and are legal under capture, and
      // first-use module loading inside a thread-local capture is permitted (every GPU test captures in a fresh process)
      cudaGraph_t g = nullptr;
      FR_CUDA_TRY(cudaStreamBeginCapture(stream, cudaStreamCaptureModeThreadLocal));
      int nk = 0;
      try {
        nk = enqueue_step();
      } catch (...) {
        cudaStreamEndCapture(stream, &g);
        if (g) cudaGraphDestroy(g);
        throw;
      }
      FR_CUDA_TRY(cudaStreamEndCapture(stream, &g));
      cudaError_t e = cudaGraphInstantiate(&graph, g, 0);
      cudaGraphDestroy(g);
      FR_CUDA_TRY(e);
      graph_kernels = nk;
    }
    for (long long i = 0; i < nsteps; ++i) {
      FR_CUDA_TRY(cudaGraphLaunch(graph, stream));
      launches += graph_kernels;
    }
  }

  void sync() override {
    FR_CUDA_TRY(cudaStreamSynchronize(stream));
    FR_CUDA_TRY(cudaGetLastError());
  }

  // Events between all kernels of `reps` RHS evaluations of the internal state; per-category and per-kernel means.
  void profile(int reps, double ms[4], fr_kernel_stat *out, int cap, int *nout, bool stage) override {
    FR_REQUIRE(reps > 0, "reps must be positive");
    std::vector<const T *> up(nt);
    std::vector<StageArgs<T>> sa(nt);
    if (stage) {
      // the variant an RK45[2R+] stage runs (both registers read and written), with zero coefficients: X and Y keep their values
      FR_CUDA_TRY(cudaStreamSynchronize(stream));
      coef_host[7] = StageCoef{0.0, 0.0};
      FR_CUDA_TRY(cudaMemcpyAsync(coef.p + 7, coef_host + 7, sizeof(StageCoef), cudaMemcpyHostToDevice, stream));
    }
    for (int t = 0; t < nt; ++t) {
      up[t] = el[t]->X.p;
      sa[t] = stage ? StageArgs<T>{coef.p + 7, el[t]->X.p, el[t]->X.p, el[t]->X.p, el[t]->Y.p}
                    : StageArgs<T>{nullptr, nullptr, nullptr, el[t]->Y.p, nullptr};
    }
    launches += run_rhs(up.data(), sa.data(), nullptr);   // warm-up
    double acc[4] = {0, 0, 0, 0};
    std::vector<fr_kernel_stat> ks;
    for (int r = 0; r < reps; ++r) {
      Timeline tl;
      tl.s = stream;
      launches += run_rhs(up.data(), sa.data(), &tl);
      FR_CUDA_TRY(cudaStreamSynchronize(stream));
      if (ks.empty()) {
        ks.resize(tl.ev.size() - 1);
        for (size_t i = 1; i < tl.ev.size(); ++i) {
          fr_kernel_stat &k = ks[i - 1];
          memset(&k, 0, sizeof(k));
          strncpy(k.name, tl.name[i].c_str(), sizeof(k.name) - 1);
          k.alg_bytes = tl.bytes[i];
          k.flops = tl.flops[i];
          k.category = tl.cat[i];
        }
      }
      for (size_t i = 1; i < tl.ev.size(); ++i) {
        float m = 0;
        cudaEventElapsedTime(&m, tl.ev[i - 1], tl.ev[i]);
        acc[tl.cat[i]] += m;
        acc[3] += m;
        ks[i - 1].ms += m / reps;
      }
      for (auto e : tl.ev) cudaEventDestroy(e);
    }
    if (ms)
      for (int i = 0; i < 4; ++i) ms[i] = acc[i] / reps;
    if (nout) *nout = (int)ks.size();
    if (out)
      for (int i = 0; i < (int)ks.size() && i < cap; ++i) out[i] = ks[i];
  }

  long long check_finite() override {
    FR_CUDA_TRY(cudaStreamSynchronize(stream));
    long long bad = 0;
    for (int t = 0; t < nt; ++t) {
      const EleView<T> &v = el[t]->view;
      std::vector<T> h((size_t)v.nupts * 5 * v.ld);
      FR_CUDA_TRY(cudaMemcpy(h.data(), el[t]->X.p, h.size() * sizeof(T), cudaMemcpyDeviceToHost));
      for (long long r = 0; r < (long long)v.nupts * 5; ++r)
        for (long long k = 0; k < v.neles; ++k) bad += std::isfinite((double)h[(size_t)r * v.ld + k]) ? 0 : 1;
    }
    return bad;
  }

  std::string describe() const override {
    std::string out;
    char line[256];
    auto add = [&](const char *type, const char *what, const PanelOp<T> &op) {
      if (!op.ok()) return;
      snprintf(line, sizeof line, "%s %s %s %dx%d %s warps=%dx%dx%d+%d NIT=%d CX=%d NE=%d stages=%dx%d B occ=%d\n", sizeof(T) == 8 ? "f64" : "f32",
               type, what, op.M, op.K, op.sparse ? "k-lists" : (op.streamed() ? "dense, streamed" : "dense"), op.NG, op.WR, op.WC, op.NG, op.NIT, op.CX, op.NE, op.nstage,
               op.stage_bytes, op.occ);
      out += line;
    };
    for (int t = 0; t < nt; ++t) {
      const EleData<T> &e = *el[t];
      if (e.pM0.pop) add(tname[t], "M0", *e.pM0.pop);
      for (int i = 0; i < e.pM0.nparts; ++i) add(tname[t], "M0/rows", *e.pM0.part[i]);
      for (auto &q : e.pGrad) add(tname[t], "[M460|M6]", q.op);
      for (auto &q : e.pDiv) add(tname[t], "[M132|M3]", q.op);
    }
    return out;
  }

  // H2D of the state (device layout, context precision), one step, D2H -- the end-to-end user call.
  void rk_step_host(double dt, void *const *u_host) override {
    FR_REQUIRE(u_host, "u_host must be non-NULL");
    for (int t = 0; t < nt; ++t) {
      FR_REQUIRE(u_host[t], "u_host[t] must be non-NULL");
      const size_t nb = (size_t)el[t]->view.nupts * 5 * el[t]->view.ld * sizeof(T);
      FR_CUDA_TRY(cudaMemcpyAsync(el[t]->X.p, u_host[t], nb, cudaMemcpyHostToDevice, stream));
    }
    rk_step(dt, 1);
    for (int t = 0; t < nt; ++t) {
      const size_t nb = (size_t)el[t]->view.nupts * 5 * el[t]->view.ld * sizeof(T);
      FR_CUDA_TRY(cudaMemcpyAsync(u_host[t], el[t]->X.p, nb, cudaMemcpyDeviceToHost, stream));
    }
    FR_CUDA_TRY(cudaStreamSynchronize(stream));
  }
};

// one line per launch of a stand-alone operator-product plan (fr_gemm_plan_describe)
template <typename T>
std::string gemm_plan_describe(const GemmPlan<T> &p) {
  std::string out;
  char line[256];
  auto add = [&](const PanelOp<T> &op, int row0) {
    snprintf(line, sizeof line, "%s rows %d..%d of %dx%d %s warps=%dx%dx%d+%d NIT=%d CX=%d NE=%d chunks=%d stages=%dx%d B\n", sizeof(T) == 8 ? "f64" : "f32",
             row0, row0 + op.M - 1, p.M, p.K, op.sparse ? "k-lists" : (op.streamed() ? "dense, streamed" : "dense"), op.NG, op.WR, op.WC, op.NG,
             op.NIT, op.CX, op.NE, op.nchunks, op.nstage, op.stage_bytes);
    out += line;
  };
  if (p.pop) add(*p.pop, 0);
  for (int i = 0; i < p.nparts; ++i) add(*p.part[i], p.part_row0[i]);
  if (!p.pop && p.nparts == 0) {
    snprintf(line, sizeof line, "%s %dx%d register-tile kernel TY=%d MT=%d row blocks=%d %s\n", sizeof(T) == 8 ? "f64" : "f32", p.M, p.K, p.TY, p.MT,
             p.nrb, p.resident ? "operator resident" : "operator streamed by cp.async");
    out += line;
  }
  return out;
}

}  // namespace frb

// ---------------------------------------------------------------------------- C ABI
struct fr_ctx {
  frb::CtxBase *impl;
};
struct fr_gemm_plan {
  fr_prec prec;
  frb::GemmPlan<double> pd;
  frb::GemmPlan<float> pf;
};

namespace {
template <typename F>
fr_status guard(std::string *err, F &&f) {
  try {
    f();
    return FR_OK;
  } catch (const frb::Error &e) {
    if (err) *err = e.msg;
    frb::g_error = e.msg;
    return e.st;
  } catch (const std::bad_alloc &) {
    if (err) *err = "host allocation failed";
    frb::g_error = "host allocation failed";
    return FR_ENOMEM;
  } catch (...) {
    if (err) *err = "unknown error";
    frb::g_error = "unknown error";
    return FR_ESTATE;
  }
}
void require_device() {
  int n = 0;
  cudaError_t e = cudaGetDeviceCount(&n);
  if (e != cudaSuccess || n <= 0)
    throw frb::Error{FR_ECUDA, std::string("no usable CUDA device: ") + (e != cudaSuccess ? cudaGetErrorString(e) : "count = 0")};
}
}  // namespace

extern "C" {

fr_status fr_setup(const fr_config *cfg, fr_ctx **out) {
  if (out) *out = nullptr;
  return guard(nullptr, [&] {
    FR_REQUIRE(cfg && out, "cfg and out must be non-NULL");
    FR_REQUIRE(cfg->prec == FR_F32 || cfg->prec == FR_F64, "prec must be FR_F32 or FR_F64");
    FR_REQUIRE(cfg->system == FR_EULER || cfg->system == FR_NAVIER_STOKES, "unknown system");
    FR_REQUIRE(cfg->stepper == FR_RK4 || cfg->stepper == FR_RK45_2R || cfg->stepper == FR_EULER1, "unknown stepper");
    FR_REQUIRE(cfg->mode == FR_MODE_FUSED || cfg->mode == FR_MODE_UNFUSED, "unknown mode");
    require_device();
    std::unique_ptr<frb::CtxBase> impl;
    if (cfg->prec == FR_F64) {
      auto c = std::make_unique<frb::Ctx<double>>();
      c->setup(cfg);
      impl = std::move(c);
    } else {
      auto c = std::make_unique<frb::Ctx<float>>();
      c->setup(cfg);
      impl = std::move(c);
    }
    *out = new fr_ctx{impl.release()};
  });
}

#define FR_CTX_CALL(ctx, body)                            \
  if (!(ctx) || !(ctx)->impl) return FR_EINVAL;           \
  return guard(&(ctx)->impl->err, [&] { body; })

fr_status fr_state_layout(const fr_ctx *ctx, int32_t et, int64_t *ld, int64_t *nbytes) {
  FR_CTX_CALL(ctx, ctx->impl->state_layout(et, ld, nbytes));
}
fr_status fr_rhs(fr_ctx *ctx, const void *const *u_dev, void *const *dudt_dev) { FR_CTX_CALL(ctx, ctx->impl->rhs(u_dev, dudt_dev)); }
fr_status fr_set_state(fr_ctx *ctx, const double *const *u_host) { FR_CTX_CALL(ctx, ctx->impl->set_state(u_host)); }
fr_status fr_get_state(fr_ctx *ctx, double *const *u_host) { FR_CTX_CALL(ctx, ctx->impl->get_state(u_host)); }
fr_status fr_rk_step(fr_ctx *ctx, double dt) { FR_CTX_CALL(ctx, ctx->impl->rk_step(dt, 1)); }
fr_status fr_rk_run(fr_ctx *ctx, double dt, int64_t nsteps) { FR_CTX_CALL(ctx, ctx->impl->rk_step(dt, nsteps)); }
fr_status fr_rk_adaptive_run(fr_ctx *ctx, double t0, double t1, double dt_init, double atol, double rtol, int64_t max_attempts,
                             fr_adapt_stats *stats, double *dt_hist, double *err_hist, int64_t hist_cap) {
  FR_CTX_CALL(ctx, ctx->impl->rk_adaptive(t0, t1, dt_init, atol, rtol, max_attempts, stats, dt_hist, err_hist, hist_cap));
}
fr_status fr_sync(fr_ctx *ctx) { FR_CTX_CALL(ctx, ctx->impl->sync()); }
fr_status fr_profile_rhs(fr_ctx *ctx, int32_t reps, double ms[4]) {
  FR_CTX_CALL(ctx, {
    FR_REQUIRE(ms, "ms must be non-NULL");
    ctx->impl->profile(reps, ms, nullptr, 0, nullptr);
  });
}
fr_status fr_profile_kernels(fr_ctx *ctx, int32_t reps, fr_kernel_stat *out, int32_t cap, int32_t *n) {
  FR_CTX_CALL(ctx, {
    FR_REQUIRE(n && (out || cap == 0), "n must be non-NULL (and out non-NULL when cap > 0)");
    int nn = 0;
    ctx->impl->profile(reps, nullptr, out, cap, &nn);
    *n = nn;
  });
}
fr_status fr_profile_stage_kernels(fr_ctx *ctx, int32_t reps, fr_kernel_stat *out, int32_t cap, int32_t *n) {
  FR_CTX_CALL(ctx, {
    FR_REQUIRE(n && (out || cap == 0), "n must be non-NULL (and out non-NULL when cap > 0)");
    int nn = 0;
    ctx->impl->profile(reps, nullptr, out, cap, &nn, true);
    *n = nn;
  });
}
fr_status fr_check_finite(fr_ctx *ctx, int64_t *n_nonfinite) {
  FR_CTX_CALL(ctx, {
    FR_REQUIRE(n_nonfinite, "n_nonfinite must be non-NULL");
    *n_nonfinite = ctx->impl->check_finite();
  });
}
fr_status fr_plan_describe(const fr_ctx *ctx, char *buf, int64_t cap) {
  if (!ctx || !ctx->impl) return FR_EINVAL;
  return guard(nullptr, [&] {
    FR_REQUIRE(buf && cap > 0, "buf must be non-NULL and cap positive");
    const std::string d = ctx->impl->describe();
    const size_t nc = std::min<size_t>(d.size(), (size_t)cap - 1);
    memcpy(buf, d.data(), nc);
    buf[nc] = 0;
  });
}
fr_status fr_rhs_phase(fr_ctx *ctx, int32_t phase, const void *const *u_dev, void *const *dudt_dev) {
  FR_CTX_CALL(ctx, ctx->impl->rhs_phase(phase, u_dev, dudt_dev));
}
fr_status fr_rk_stage_phase(fr_ctx *ctx, double dt, int32_t stage, int32_t phase) { FR_CTX_CALL(ctx, ctx->impl->rk_stage_phase(dt, stage, phase)); }
fr_status fr_halo_buffers(fr_ctx *ctx, int32_t which, void **send_dev, void **recv_dev, int64_t *nvalues) {
  FR_CTX_CALL(ctx, ctx->impl->halo_buffers(which, send_dev, recv_dev, nvalues));
}
fr_status fr_halo_set_peers(fr_ctx *ctx, int32_t npeers, const int64_t *start, const int64_t *count) {
  FR_CTX_CALL(ctx, ctx->impl->halo_set_peers(npeers, start, count));
}
fr_status fr_rk_step_host(fr_ctx *ctx, double dt, void *const *u_host) { FR_CTX_CALL(ctx, ctx->impl->rk_step_host(dt, u_host)); }
int64_t fr_launch_count(const fr_ctx *ctx) { return ctx && ctx->impl ? ctx->impl->launches : 0; }
const char *fr_last_error(const fr_ctx *ctx) { return ctx && ctx->impl ? ctx->impl->err.c_str() : "invalid context"; }
const char *fr_global_error(void) { return frb::g_error.c_str(); }
void fr_destroy(fr_ctx *ctx) {
  if (!ctx) return;
  delete ctx->impl;
  delete ctx;
}

fr_status fr_gemm_plan_create(int32_t M, int32_t K, const double *A_host, fr_prec prec, fr_gemm_plan **out) {
  if (out) *out = nullptr;
  return guard(nullptr, [&] {
    FR_REQUIRE(out, "out must be non-NULL");
    FR_REQUIRE(prec == FR_F32 || prec == FR_F64, "prec must be FR_F32 or FR_F64");
    require_device();
    auto p = std::make_unique<fr_gemm_plan>();
    p->prec = prec;
    if (prec == FR_F64) {
      frb::gemm_plan_build(p->pd, M, K, A_host, 0.0);
      frb::gemm_plan_tune(p->pd, A_host, 0.0);
    } else {
      frb::gemm_plan_build(p->pf, M, K, A_host, 0.0);
      frb::gemm_plan_tune(p->pf, A_host, 0.0);
    }
    *out = p.release();
  });
}
fr_status fr_gemm_plan_run(fr_gemm_plan *plan, int64_t N, double c1, const void *B_dev, int64_t ldb, double c2, void *C_dev,
                           int64_t ldc, void *cuda_stream) {
  return guard(nullptr, [&] {
    FR_REQUIRE(plan && B_dev && C_dev, "plan, B and C must be non-NULL");
    FR_REQUIRE(N >= 0, "N must be >= 0");
    cudaStream_t s = (cudaStream_t)cuda_stream;
    if (plan->prec == FR_F64)
      frb::gemm_run(plan->pd, N, c1, (const double *)B_dev, ldb, 0, c2, (double *)C_dev, ldc, 0, 1, s);
    else
      frb::gemm_run(plan->pf, N, (float)c1, (const float *)B_dev, ldb, 0, (float)c2, (float *)C_dev, ldc, 0, 1, s);
  });
}
fr_status fr_gemm_plan_describe(const fr_gemm_plan *plan, char *buf, int64_t cap) {
  return guard(nullptr, [&] {
    FR_REQUIRE(plan && buf && cap > 0, "plan and buf must be non-NULL and cap positive");
    const std::string d = plan->prec == FR_F64 ? frb::gemm_plan_describe(plan->pd) : frb::gemm_plan_describe(plan->pf);
    const size_t nc = std::min<size_t>(d.size(), (size_t)cap - 1);
    memcpy(buf, d.data(), nc);
    buf[nc] = 0;
  });
}
void fr_gemm_plan_destroy(fr_gemm_plan *plan) {
  if (!plan) return;
  frb::gemm_plan_free(plan->pd);
  frb::gemm_plan_free(plan->pf);
  delete plan;
}
fr_status fr_gemm(int32_t M, int32_t K, int64_t N, double c1, const double *A_host, const void *B_dev, int64_t ldb, double c2,
                  void *C_dev, int64_t ldc, fr_prec prec, void *cuda_stream) {
  // a one-shot product takes the statically best geometry: timing candidates would cost more than the product
  fr_gemm_plan *p = nullptr;
  fr_status st = guard(nullptr, [&] {
    FR_REQUIRE(prec == FR_F32 || prec == FR_F64, "prec must be FR_F32 or FR_F64");
    require_device();
    auto q = std::make_unique<fr_gemm_plan>();
    q->prec = prec;
    if (prec == FR_F64) frb::gemm_plan_build(q->pd, M, K, A_host, 0.0);
    else frb::gemm_plan_build(q->pf, M, K, A_host, 0.0);
    p = q.release();
  });
  if (st != FR_OK) return st;
  st = fr_gemm_plan_run(p, N, c1, B_dev, ldb, c2, C_dev, ldc, cuda_stream);
  if (st == FR_OK) {
    // the operator buffer is freed below: wait for the product that reads it
    cudaError_t e = cudaStreamSynchronize((cudaStream_t)cuda_stream);
    if (e != cudaSuccess) {
      frb::g_error = std::string("fr_gemm: ") + cudaGetErrorString(e);
      st = FR_ECUDA;
    }
  }
  fr_gemm_plan_destroy(p);
  return st;
}
fr_status fr_gemm_static(int32_t M, int32_t K, int64_t N, double c1, const double *A_host, const void *B_dev, int64_t ldb, double c2,
                         void *C_dev, int64_t ldc, fr_prec prec, void *cuda_stream) {
  return guard(nullptr, [&] {
    FR_REQUIRE(prec == FR_F32 || prec == FR_F64, "prec must be FR_F32 or FR_F64");
    require_device();
    cudaStream_t s = (cudaStream_t)cuda_stream;
    if (prec == FR_F64) frb::gemm_static_run<double>(M, K, N, c1, A_host, (const double *)B_dev, ldb, c2, (double *)C_dev, ldc, s);
    else frb::gemm_static_run<float>(M, K, N, (float)c1, A_host, (const float *)B_dev, ldb, (float)c2, (float *)C_dev, ldc, s);
  });
}

}  // extern "C"
