// Point-wise kernels of the unfused chain: one kernel per step S2, S4, S6, S7, S9/S10 of SURVEY 8(a)
// ("point-wise, concerning themselves solely with data at an individual solution/flux point").
// All arrays are SoA with the element index fastest, so a warp reads / writes 32 consecutive elements.
#include "kernels.cuh"
#include "physics.cuh"

namespace frb {

namespace {

constexpr int PW_BLOCK = 128;

template <typename T>
__device__ __forceinline__ void load_smats(const T *smats, int affine, int nupts, int rho, long long ld, long long e,
                                           T S[3][3]) {
#pragma unroll
  for (int a = 0; a < 3; ++a)
#pragma unroll
    for (int i = 0; i < 3; ++i)
      S[a][i] = affine ? smats[(long long)(a * 3 + i) * ld + e] : smats[((long long)(a * 3 + i) * nupts + rho) * ld + e];
}

// S6: F~_alpha = sum_i S[alpha][i] (f^inv_i(U) - f^visc_i(U, G)); G (if NS) is overwritten in place by F~.
template <typename T>
__global__ void __launch_bounds__(PW_BLOCK) k_tdisf(EleView<T> ev, const T *__restrict__ u, T *gf, PhysParams<T> ph) {
  // Affine types (one set of metric terms per element): a 1-D grid with the solution point fastest, so that the blocks that share
  // an element range -- and its metric terms -- run back to back and re-read them from L1 / L2, not from DRAM (with the point
  // slowest the 26 MB of FP64 terms of config 3's tetrahedra came back from DRAM several times: 1.15x the algorithmic bytes).
  long long eb = blockIdx.x;
  int rho = blockIdx.y;
  if (ev.affine) {
    rho = (int)(eb % ev.nupts);
    eb /= ev.nupts;
  }
  const long long e = eb * PW_BLOCK + threadIdx.x;
  if (e >= ev.ld) return;
  const long long ld = ev.ld;
  T out[3][5];
  if (e < ev.neles) {
    T uu[5];
#pragma unroll
    for (int v = 0; v < 5; ++v) uu[v] = u[((long long)rho * 5 + v) * ld + e];
    T f[3][5], rr, vel[3], p;
    inviscid_flux(uu, ph.gamma, f, rr, vel, p);
    if (ph.ns) {
      T q[3][5];
#pragma unroll
      for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int v = 0; v < 5; ++v) q[i][v] = gf[(((long long)i * ev.nupts + rho) * 5 + v) * ld + e];
      subtract_viscous_flux(uu, q, rr, vel, ph.gamma, ph.mu, ph.prandtl, f);
    }
    T S[3][3];
    load_smats(ev.smats, ev.affine, ev.nupts, rho, ld, e, S);
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
      for (int v = 0; v < 5; ++v) out[a][v] = S[a][0] * f[0][v] + S[a][1] * f[1][v] + S[a][2] * f[2][v];
  } else {
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
      for (int v = 0; v < 5; ++v) out[a][v] = T(0);
  }
#pragma unroll
  for (int a = 0; a < 3; ++a)
#pragma unroll
    for (int v = 0; v < 5; ++v) gf[(((long long)a * ev.nupts + rho) * 5 + v) * ld + e] = out[a][v];
}

// S4: physical gradient G_i = (1/|J|) sum_alpha S[alpha][i] G~_alpha, in place.
template <typename T>
__global__ void __launch_bounds__(PW_BLOCK) k_gradcoru(EleView<T> ev, T *g) {
  const long long e = (long long)blockIdx.x * PW_BLOCK + threadIdx.x;
  const int rho = blockIdx.y;
  if (e >= ev.ld) return;
  const long long ld = ev.ld;
  T out[3][5];
  if (e < ev.neles) {
    T S[3][3];
    load_smats(ev.smats, ev.affine, ev.nupts, rho, ld, e, S);
    const T rj = ev.affine ? ev.rcpdjac[e] : ev.rcpdjac[(long long)rho * ld + e];
    T gt[3][5];
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
      for (int v = 0; v < 5; ++v) gt[a][v] = g[(((long long)a * ev.nupts + rho) * 5 + v) * ld + e];
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
      for (int v = 0; v < 5; ++v) out[i][v] = rj * (S[0][i] * gt[0][v] + S[1][i] * gt[1][v] + S[2][i] * gt[2][v]);
  } else {
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
      for (int v = 0; v < 5; ++v) out[i][v] = T(0);
  }
#pragma unroll
  for (int i = 0; i < 3; ++i)
#pragma unroll
    for (int v = 0; v < 5; ++v) g[(((long long)i * ev.nupts + rho) * 5 + v) * ld + e] = out[i][v];
}

// S9 (+S10): K = -R/|J|;  plain: out1 = K;  stage update: out1 = in1 + c1 K, out2 = in2 + c2 K.
template <typename T>
__global__ void __launch_bounds__(PW_BLOCK) k_negdivconf(EleView<T> ev, const T *__restrict__ r, StageArgs<T> sa) {
  const long long e = (long long)blockIdx.x * PW_BLOCK + threadIdx.x;
  const int rho = blockIdx.y;
  if (e >= ev.ld) return;
  const long long ld = ev.ld;
  const bool live = e < ev.neles;
  const T rj = live ? (ev.affine ? ev.rcpdjac[e] : ev.rcpdjac[(long long)rho * ld + e]) : T(0);
  T c1 = T(0), c2 = T(0);
  if (sa.coef) {
    c1 = (T)sa.coef->c1;
    c2 = (T)sa.coef->c2;
  }
#pragma unroll
  for (int v = 0; v < 5; ++v) {
    const long long idx = ((long long)rho * 5 + v) * ld + e;
    const T k = live ? -r[idx] * rj : T(0);
    if (!sa.coef) {
      sa.out1[idx] = k;
    } else {
      const T a = sa.in1[idx], b = sa.in2 ? sa.in2[idx] : T(0);
      sa.out1[idx] = live ? a + c1 * k : T(0);
      if (sa.out2) sa.out2[idx] = live ? b + c2 * k : T(0);
    }
  }
}

template <typename T>
__device__ __forceinline__ void side_addr(const TypeTab &tt, int e, int ts, long long &uoff, long long &goff,
                                          long long &ld, long long &gcomp) {
  const int t = ts >> 16, sig = ts & 0xffff;
  ld = tt.ld[t];
  const long long rel = (long long)sig * 5 * ld + e;
  uoff = tt.ubase[t] + rel;
  goff = tt.gbase[t] + rel;
  gcomp = tt.gcomp[t];
}

// S2: common solution C = (1/2 - beta) u_L + (1/2 + beta) u_R, stored at both flux points.
// jump != 0: store the correction C - u_own instead (the fused gradient kernel then applies [M4 | M6] to [U; C - U_f], which equals
// [M460 | M6][U; C] because M460 = M4 - M6 M0).  With beta = 1/2 the correction vanishes on the R side, whose entries stay at their
// initial zero and are never written: the scattered R-side store of this kernel disappears.
template <typename T>
__global__ void __launch_bounds__(PW_BLOCK) k_con_u(IfaceView<T> iv, const __grid_constant__ TypeTab tt,
                                                    const T *__restrict__ uf, T *cf, T beta, int jump) {
  const long long k = (long long)blockIdx.x * PW_BLOCK + threadIdx.x;
  if (k >= iv.npairs) return;
  const PairRec pr = iv.pairs[k];
  long long ul, gl, ldl, gcl, ur, gr, ldr, gcr;
  side_addr<T>(tt, pr.le, pr.lts, ul, gl, ldl, gcl);
  side_addr<T>(tt, pr.re, pr.rts, ur, gr, ldr, gcr);
  const T wl = T(0.5) - beta, wr = T(0.5) + beta;
  if (jump) {
#pragma unroll
    for (int v = 0; v < 5; ++v) {
      const T d = uf[ur + v * ldr] - uf[ul + v * ldl];
      cf[ul + v * ldl] = wr * d;
      if (wl != T(0)) cf[ur + v * ldr] = -wl * d;
    }
    return;
  }
  if (wl == T(0)) {
    // beta = 1/2 (the default, reading R9): C = u_R on both sides, the L state is not needed
#pragma unroll
    for (int v = 0; v < 5; ++v) {
      const T c = wr * uf[ur + v * ldr];
      cf[ul + v * ldl] = c;
      cf[ur + v * ldr] = c;
    }
    return;
  }
#pragma unroll
  for (int v = 0; v < 5; ++v) {
    const T c = wl * uf[ul + v * ldl] + wr * uf[ur + v * ldr];
    cf[ul + v * ldl] = c;
    cf[ur + v * ldr] = c;
  }
}

// S7: common normal flux (Rusanov + LDG viscous + penalty) times the per-side magnitude, written in place over
// U_f with opposite signs (each flux point is read and written by exactly one thread).
// LONLY: beta = 1/2 (the default, reading R9): the viscous part takes the L side's gradient alone.  A compile-time variant, so that the
// R-side gradient, its weights and its branch take no registers: FP64 167 -> 120 (four CTAs per SM instead of three), FP32 102 -> 79
// (six instead of four); S7 is latency-bound below its DRAM rate, and ran 11 % / 17 % faster.  Forcing more CTAs per SM by launch
// bounds (96 / 80 / 64 registers) spills and is slower.
template <typename T, bool LONLY>
__global__ void __launch_bounds__(PW_BLOCK) k_comm_flux(IfaceView<T> iv, const __grid_constant__ TypeTab tt, T *uf,
                                                        const T *__restrict__ gf, PhysParams<T> ph) {
  const long long k = (long long)blockIdx.x * PW_BLOCK + threadIdx.x;
  if (k >= iv.npairs) return;
  const PairRec pr = iv.pairs[k];
  long long ul, gl, ldl, gcl, ur, gr, ldr, gcr;
  side_addr<T>(tt, pr.le, pr.lts, ul, gl, ldl, gcl);
  side_addr<T>(tt, pr.re, pr.rts, ur, gr, ldr, gcr);
  T uL[5], uR[5], qL[3][5], qR[3][5];
#pragma unroll
  for (int v = 0; v < 5; ++v) {
    uL[v] = uf[ul + v * ldl];
    uR[v] = uf[ur + v * ldr];
  }
  const T wL = LONLY ? T(1) : T(0.5) + ph.beta, wR = LONLY ? T(0) : T(0.5) - ph.beta;
  if (ph.ns) {
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
      for (int v = 0; v < 5; ++v) {
        qL[i][v] = (LONLY || wL != T(0)) ? gf[gl + i * gcl + v * ldl] : T(0);
        qR[i][v] = (!LONLY && wR != T(0)) ? gf[gr + i * gcr + v * ldr] : T(0);
      }
  }
  const T n[3] = {iv.nl[k], iv.nl[iv.npairs + k], iv.nl[2 * iv.npairs + k]};
  T F[5];
  common_flux(uL, uR, uL, qL, uR, qR, uR, n, ph, wL, wR, F);
  const T ml = iv.magl[k], mr = iv.magr[k];
#pragma unroll
  for (int v = 0; v < 5; ++v) {
    uf[ul + v * ldl] = ml * F[v];
    uf[ur + v * ldr] = -mr * F[v];
  }
}

template <typename T>
__device__ __forceinline__ void bc_states(int type, const T uL[5], const T n[3], T gamma, const T *par, T ub[5],
                                          T uv[5]) {
  if (type == FR_BC_NOSLIP_ISOTHERMAL_WALL) {
    ghost_wall(uL, par[0], ub, uv);
  } else {
    ghost_farfield(uL, n, gamma, par, ub);
#pragma unroll
    for (int v = 0; v < 5; ++v) uv[v] = ub[v];
  }
}

// S2 at boundary flux points: C = u_visc(u_L).
template <typename T>
__global__ void __launch_bounds__(PW_BLOCK) k_bc_con_u(BndView<T> bv, const __grid_constant__ TypeTab tt,
                                                       const T *__restrict__ uf, T *cf, T gamma, int jump) {
  const long long k = (long long)blockIdx.x * PW_BLOCK + threadIdx.x;
  if (k >= bv.n) return;
  const BndRec br = bv.recs[k];
  long long ul, gl, ldl, gcl;
  side_addr<T>(tt, br.e, br.ts, ul, gl, ldl, gcl);
  T uL[5], ub[5], uv[5];
#pragma unroll
  for (int v = 0; v < 5; ++v) uL[v] = uf[ul + v * ldl];
  const T n[3] = {bv.nrm[k], bv.nrm[bv.n + k], bv.nrm[2 * bv.n + k]};
  bc_states(bv.type, uL, n, gamma, bv.par, ub, uv);
#pragma unroll
  for (int v = 0; v < 5; ++v) cf[ul + v * ldl] = jump ? uv[v] - uL[v] : uv[v];
}

// S7 at boundary flux points: ghost state as u_R, G_f,R := G_f,L, only D_L stored.
template <typename T>
__global__ void __launch_bounds__(PW_BLOCK) k_bc_comm_flux(BndView<T> bv, const __grid_constant__ TypeTab tt, T *uf,
                                                           const T *__restrict__ gf, PhysParams<T> ph) {
  const long long k = (long long)blockIdx.x * PW_BLOCK + threadIdx.x;
  if (k >= bv.n) return;
  const BndRec br = bv.recs[k];
  long long ul, gl, ldl, gcl;
  side_addr<T>(tt, br.e, br.ts, ul, gl, ldl, gcl);
  T uL[5], ub[5], uv[5], qL[3][5];
#pragma unroll
  for (int v = 0; v < 5; ++v) uL[v] = uf[ul + v * ldl];
  if (ph.ns) {
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
      for (int v = 0; v < 5; ++v) qL[i][v] = gf[gl + i * gcl + v * ldl];
  }
  const T n[3] = {bv.nrm[k], bv.nrm[bv.n + k], bv.nrm[2 * bv.n + k]};
  bc_states(bv.type, uL, n, ph.gamma, bv.par, ub, uv);
  T F[5];
  common_flux(uL, ub, uv, qL, uv, qL, uv, n, ph, T(1), T(0), F);
  const T m = bv.mag[k];
#pragma unroll
  for (int v = 0; v < 5; ++v) uf[ul + v * ldl] = m * F[v];
}

inline unsigned blocks_for(long long n) { return (unsigned)((n + PW_BLOCK - 1) / PW_BLOCK); }

}  // namespace

template <typename T>
int launch_tdisf(const EleView<T> &ev, const T *u, T *gf, const PhysParams<T> &ph, cudaStream_t s) {
  dim3 grid(blocks_for(ev.ld), ev.nupts);
  if (ev.affine) grid = dim3((unsigned)((long long)blocks_for(ev.ld) * ev.nupts), 1);
  k_tdisf<T><<<grid, PW_BLOCK, 0, s>>>(ev, u, gf, ph);
  FR_CUDA_TRY(cudaGetLastError());
  return 1;
}
template <typename T>
int launch_gradcoru(const EleView<T> &ev, T *g, cudaStream_t s) {
  dim3 grid(blocks_for(ev.ld), ev.nupts);
  k_gradcoru<T><<<grid, PW_BLOCK, 0, s>>>(ev, g);
  FR_CUDA_TRY(cudaGetLastError());
  return 1;
}
template <typename T>
int launch_negdivconf(const EleView<T> &ev, const T *r, const StageArgs<T> &sa, cudaStream_t s) {
  dim3 grid(blocks_for(ev.ld), ev.nupts);
  k_negdivconf<T><<<grid, PW_BLOCK, 0, s>>>(ev, r, sa);
  FR_CUDA_TRY(cudaGetLastError());
  return 1;
}
template <typename T>
int launch_con_u(const IfaceView<T> &iv, const TypeTab &tt, const T *uf, T *cf, T beta, int jump, cudaStream_t s) {
  if (iv.npairs == 0) return 0;
  k_con_u<T><<<blocks_for(iv.npairs), PW_BLOCK, 0, s>>>(iv, tt, uf, cf, beta, jump);
  FR_CUDA_TRY(cudaGetLastError());
  return 1;
}
template <typename T>
int launch_comm_flux(const IfaceView<T> &iv, const TypeTab &tt, T *uf, const T *gf, const PhysParams<T> &ph,
                     cudaStream_t s) {
  if (iv.npairs == 0) return 0;
  if (ph.ns && ph.beta == T(0.5)) k_comm_flux<T, true><<<blocks_for(iv.npairs), PW_BLOCK, 0, s>>>(iv, tt, uf, gf, ph);
  else k_comm_flux<T, false><<<blocks_for(iv.npairs), PW_BLOCK, 0, s>>>(iv, tt, uf, gf, ph);
  FR_CUDA_TRY(cudaGetLastError());
  return 1;
}
template <typename T>
int launch_bc_con_u(const BndView<T> &bv, const TypeTab &tt, const T *uf, T *cf, T gamma, int jump, cudaStream_t s) {
  if (bv.n == 0) return 0;
  k_bc_con_u<T><<<blocks_for(bv.n), PW_BLOCK, 0, s>>>(bv, tt, uf, cf, gamma, jump);
  FR_CUDA_TRY(cudaGetLastError());
  return 1;
}
template <typename T>
int launch_bc_comm_flux(const BndView<T> &bv, const TypeTab &tt, T *uf, const T *gf, const PhysParams<T> &ph,
                        cudaStream_t s) {
  if (bv.n == 0) return 0;
  k_bc_comm_flux<T><<<blocks_for(bv.n), PW_BLOCK, 0, s>>>(bv, tt, uf, gf, ph);
  FR_CUDA_TRY(cudaGetLastError());
  return 1;
}

// ---- halo exchange: pack the own values at the cut flux points / unpack the received ones into the ghost flux points
template <typename T>
__global__ void __launch_bounds__(PW_BLOCK) k_halo_pack(HaloView hv, int ncomp, const T *__restrict__ src, T *__restrict__ send) {
  const long long i = (long long)blockIdx.x * PW_BLOCK + threadIdx.x;
  if (i >= hv.n) return;
  const long long off = ncomp == 1 ? hv.off_u[i] : hv.off_g[i], ld = hv.ld[i], gc = hv.gcomp[i];
  const long long cnt = hv.pcnt[i];
  T *d = send + 5ll * ncomp * hv.pstart[i] + hv.pj[i];
  for (int c = 0; c < ncomp; ++c)
#pragma unroll
    for (int v = 0; v < 5; ++v) d[(5 * c + v) * cnt] = src[off + c * gc + v * ld];
}
template <typename T>
__global__ void __launch_bounds__(PW_BLOCK) k_halo_unpack(HaloView hv, int ncomp, const T *__restrict__ recv, T *__restrict__ dst) {
  const long long i = (long long)blockIdx.x * PW_BLOCK + threadIdx.x;
  if (i >= hv.n) return;
  const long long cnt = hv.pcnt[i];
  const T *r = recv + 5ll * ncomp * hv.pstart[i] + hv.pj[i];
  T *d = dst + (ncomp == 1 ? hv.ghost_u : hv.ghost_g) + i;
  for (int c = 0; c < ncomp; ++c)
#pragma unroll
    for (int v = 0; v < 5; ++v) d[c * hv.ghost_gcomp + v * hv.ghost_ld] = r[(5 * c + v) * cnt];
}
template <typename T>
int launch_halo_pack(const HaloView &hv, int which, const T *src, T *send, cudaStream_t s) {
  if (hv.n == 0) return 0;
  k_halo_pack<T><<<(unsigned)((hv.n + PW_BLOCK - 1) / PW_BLOCK), PW_BLOCK, 0, s>>>(hv, which ? 3 : 1, src, send);
  FR_CUDA_TRY(cudaGetLastError());
  return 1;
}
template <typename T>
int launch_halo_unpack(const HaloView &hv, int which, const T *recv, T *dst, cudaStream_t s) {
  if (hv.n == 0) return 0;
  k_halo_unpack<T><<<(unsigned)((hv.n + PW_BLOCK - 1) / PW_BLOCK), PW_BLOCK, 0, s>>>(hv, which ? 3 : 1, recv, dst);
  FR_CUDA_TRY(cudaGetLastError());
  return 1;
}

#define FR_INST(T)                                                                                              \
  template int launch_tdisf<T>(const EleView<T> &, const T *, T *, const PhysParams<T> &, cudaStream_t);       \
  template int launch_gradcoru<T>(const EleView<T> &, T *, cudaStream_t);                                      \
  template int launch_negdivconf<T>(const EleView<T> &, const T *, const StageArgs<T> &, cudaStream_t);        \
  template int launch_con_u<T>(const IfaceView<T> &, const TypeTab &, const T *, T *, T, int, cudaStream_t);        \
  template int launch_comm_flux<T>(const IfaceView<T> &, const TypeTab &, T *, const T *, const PhysParams<T> &, \
                                   cudaStream_t);                                                               \
  template int launch_bc_con_u<T>(const BndView<T> &, const TypeTab &, const T *, T *, T, int, cudaStream_t);       \
  template int launch_bc_comm_flux<T>(const BndView<T> &, const TypeTab &, T *, const T *, const PhysParams<T> &, \
                                      cudaStream_t);                                                            \
  template int launch_halo_pack<T>(const HaloView &, int, const T *, T *, cudaStream_t);                       \
  template int launch_halo_unpack<T>(const HaloView &, int, const T *, T *, cudaStream_t);
FR_INST(double)
FR_INST(float)

}  // namespace frb
