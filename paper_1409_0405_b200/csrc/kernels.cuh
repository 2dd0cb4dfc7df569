// Device-side views and kernel launchers shared by the stage driver (api.cu).
#pragma once
#include "common.cuh"
#include "panel.cuh"

namespace frb {

// One element type on the device (all arrays in precision T, element index fastest, leading dimension ld).
template <typename T>
struct EleView {
  int nupts, nfpts, affine;
  long long neles, ld;
  const T *smats;     // [3][3][nupts][ld]  or [3][3][ld] if affine
  const T *rcpdjac;   // [nupts][ld]        or [ld] if affine
};

template <typename T>
struct IfaceView {
  long long npairs;
  const PairRec *pairs;
  const T *nl;        // [3][npairs]
  const T *magl, *magr;
};

template <typename T>
struct BndView {
  long long n;
  int type;
  const BndRec *recs;
  const T *nrm;       // [3][n]
  const T *mag;
  T par[8];
};

// Fused Runge-Kutta stage update (S10): out1 = in1 + c1*K, out2 = in2 + c2*K with K = -R/|J|.
// coef == nullptr: plain S9, out1 = K.
template <typename T>
struct StageArgs {
  const StageCoef *coef;
  const T *in1, *in2;
  T *out1, *out2;
};

template <typename T>
int launch_tdisf(const EleView<T> &ev, const T *u, T *gf, const PhysParams<T> &ph, cudaStream_t s);
template <typename T>
int launch_gradcoru(const EleView<T> &ev, T *g, cudaStream_t s);
template <typename T>
int launch_negdivconf(const EleView<T> &ev, const T *r, const StageArgs<T> &sa, cudaStream_t s);
template <typename T>
int launch_con_u(const IfaceView<T> &iv, const TypeTab &tt, const T *uf, T *cf, T beta, int jump, cudaStream_t s);
template <typename T>
int launch_comm_flux(const IfaceView<T> &iv, const TypeTab &tt, T *uf, const T *gf, const PhysParams<T> &ph,
                     cudaStream_t s);
template <typename T>
int launch_bc_con_u(const BndView<T> &bv, const TypeTab &tt, const T *uf, T *cf, T gamma, int jump, cudaStream_t s);
template <typename T>
int launch_bc_comm_flux(const BndView<T> &bv, const TypeTab &tt, T *uf, const T *gf, const PhysParams<T> &ph,
                        cudaStream_t s);

// Halo exchange (include/frb200.h fr_halo_desc): gather the own values at the cut flux points into the send
// buffer / scatter the received values into the ghost flux points.  Entry i: own flux point at src[off[i] + c*gcomp[i] + v*ld[i]]
// (c < ncomp components of 5 variables), buffer element (5*ncomp)*pstart[i] + (5*c + v)*pcnt[i] + pj[i].
struct HaloView {
  long long n;
  const long long *off_u, *off_g, *ld, *gcomp;   // own side of every cut pair
  const long long *pstart, *pcnt, *pj;           // peer segment of entry i and its position in it
  long long ghost_u, ghost_g, ghost_ld, ghost_gcomp;   // the ghost pseudo type in the flat flux-point arrays
};
template <typename T>
int launch_halo_pack(const HaloView &hv, int which, const T *src, T *send, cudaStream_t s);
template <typename T>
int launch_halo_unpack(const HaloView &hv, int which, const T *recv, T *dst, cudaStream_t s);

// Embedded error estimate of RK45[2R+] and its norm (rk_adapt.cu)
int rk_err_blocks();
template <typename T>
int launch_rk_err_accum(T *E, const T *Y, const T *X, double g, int first, long long n, cudaStream_t s);
template <typename T>
int launch_rk_err_norm(const T *E, const T *Y, const T *X, const T *U0, double g, const double *tol_dev, long long n,
                       double *partial, cudaStream_t s);
int launch_rk_err_final(const double *partial, int n, double *out, cudaStream_t s);

// Fused panel kernels (panel_fused.cu).  *_build return false if the operator does not fit the resident design.
template <typename T>
bool fused_div_build(PanelOp<T> &op, int nu, int nf, const double *M132, const double *M3, int cand = 0, int r0 = 0, int nr = -1);
template <typename T>
int launch_fused_div(const PanelOp<T> &op, const EleView<T> &ev, const T *ftil, const T *d, const StageArgs<T> &sa,
                     cudaStream_t s);
template <typename T>
bool fused_grad_build(PanelOp<T> &op, int nu, int nf, const double *M460, const double *M6, int cand = 0, const double *M0_jump = nullptr,
                      int r0 = 0, int nr = -1);
template <typename T>
int launch_fused_grad(const PanelOp<T> &op, const EleView<T> &ev, const T *u, const T *c, T *grad, cudaStream_t s);

// Plain operator product on the panel kernels (panel_gemm.cu); `cand` as above.
// drop_rel: entries with |a| <= drop_rel * max|A| count as structural zeros (reading R24; 0 = exact zeros only)
template <typename T>
bool panel_gemm_build(PanelOp<T> &op, int M, int K, const double *A, int cand = 0, double drop_rel = 1.4210854715202004e-14, int stream = 0);
template <typename T>
void panel_gemm_run(const PanelOp<T> &op, long long N, T c1, const T *B, long long ldb, long long bsB, T c2, T *C,
                    long long ldc, long long bsC, int nbatch, cudaStream_t s);

}  // namespace frb
