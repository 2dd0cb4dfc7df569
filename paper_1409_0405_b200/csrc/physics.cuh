// Point-wise physics of the compressible Euler / Navier-Stokes equations (device functions, T = float | double).
// "All other operations involved in an FR time-step are point-wise".  Ideal gas, constant
// viscosity; formulas: DESIGN.md readings R8 (Rusanov speed), R10 (viscous flux), R11 (BCs).
#pragma once
#include "common.cuh"

namespace frb {

template <typename T>
__device__ __forceinline__ T fr_sqrt(T x) {
  return sqrt(x);
}
template <typename T>
__device__ __forceinline__ T fr_max(T a, T b) {
  return a > b ? a : b;
}

// f[i][v] = inviscid flux component i of variable v; also returns 1/rho, velocity and pressure.
template <typename T>
__device__ __forceinline__ void inviscid_flux(const T u[5], T gamma, T f[3][5], T &rrho, T v[3], T &p) {
  rrho = T(1) / u[0];
  v[0] = u[1] * rrho;
  v[1] = u[2] * rrho;
  v[2] = u[3] * rrho;
  p = (gamma - T(1)) * (u[4] - T(0.5) * (u[1] * v[0] + u[2] * v[1] + u[3] * v[2]));
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    f[i][0] = u[1 + i];
    f[i][1] = u[1 + i] * v[0];
    f[i][2] = u[1 + i] * v[1];
    f[i][3] = u[1 + i] * v[2];
    f[i][1 + i] += p;
    f[i][4] = (u[4] + p) * v[i];
  }
}

// f[i][v] -= viscous flux (Newtonian, Stokes hypothesis, Fourier heat flux, kappa = mu c_p / Pr);
// q[i][v] = d u_v / d x_i.
template <typename T>
__device__ __forceinline__ void subtract_viscous_flux(const T u[5], const T q[3][5], T rrho, const T v[3], T gamma,
                                                      T mu, T prandtl, T f[3][5]) {
  T dv[3][3];   // dv[i][j] = d_i v_j
#pragma unroll
  for (int i = 0; i < 3; ++i)
#pragma unroll
    for (int j = 0; j < 3; ++j) dv[i][j] = (q[i][1 + j] - v[j] * q[i][0]) * rrho;
  const T div = dv[0][0] + dv[1][1] + dv[2][2];
  const T Er = u[4] * rrho;
  const T kap = mu * gamma / prandtl;
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    // d_i e = (d_i E - (E/rho) d_i rho) / rho - sum_j v_j d_i v_j
    const T de = (q[i][4] - Er * q[i][0]) * rrho - (v[0] * dv[i][0] + v[1] * dv[i][1] + v[2] * dv[i][2]);
    T work = T(0);
#pragma unroll
    for (int j = 0; j < 3; ++j) {
      T tau = dv[i][j] + dv[j][i];
      if (i == j) tau -= T(2.0 / 3.0) * div;
      tau *= mu;
      f[i][1 + j] -= tau;
      work += v[j] * tau;
    }
    f[i][4] -= work + kap * de;
  }
}

// |v.n| + c
template <typename T>
__device__ __forceinline__ T wave_speed(const T u[5], const T n[3], T gamma) {
  const T rrho = T(1) / u[0];
  const T vx = u[1] * rrho, vy = u[2] * rrho, vz = u[3] * rrho;
  const T p = (gamma - T(1)) * (u[4] - T(0.5) * (u[1] * vx + u[2] * vy + u[3] * vz));
  return fabs(vx * n[0] + vy * n[1] + vz * n[2]) + fr_sqrt(gamma * p * rrho);
}

// Common normal flux at a flux point:
//   F = Rusanov(uL, uR, n) - [(1/2+beta) fv(uL,qL) + (1/2-beta) fv(uR,qR)].n + tau (uL - uR)
// For Euler (ns == 0) only the Rusanov part.  `uvL`, `uvR`: states used in the viscous fluxes (differ from
// uL / uR only at boundaries); `pen`: state subtracted in the penalty term (uR interior, u_visc at boundaries).
template <typename T>
__device__ __forceinline__ void common_flux(const T uL[5], const T uR[5], const T uvL[5], const T qL[3][5], const T uvR[5],
                                            const T qR[3][5], const T pen[5], const T n[3], const PhysParams<T> &ph,
                                            T wL, T wR, T F[5]) {
  T fL[3][5], fR[3][5], rr, vv[3], pp;
  inviscid_flux(uL, ph.gamma, fL, rr, vv, pp);
  const T cL = fabs(vv[0] * n[0] + vv[1] * n[1] + vv[2] * n[2]) + fr_sqrt(ph.gamma * pp * rr);
  inviscid_flux(uR, ph.gamma, fR, rr, vv, pp);
  const T cR = fabs(vv[0] * n[0] + vv[1] * n[1] + vv[2] * n[2]) + fr_sqrt(ph.gamma * pp * rr);
  const T lam = fr_max(cL, cR);
#pragma unroll
  for (int k = 0; k < 5; ++k)
    F[k] = T(0.5) * ((fL[0][k] + fR[0][k]) * n[0] + (fL[1][k] + fR[1][k]) * n[1] + (fL[2][k] + fR[2][k]) * n[2]) +
           T(0.5) * lam * (uL[k] - uR[k]);
  if (ph.ns) {
    T g[3][5];
    if (wL != T(0)) {
#pragma unroll
      for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int k = 0; k < 5; ++k) g[i][k] = T(0);
      const T r = T(1) / uvL[0];
      const T v3[3] = {uvL[1] * r, uvL[2] * r, uvL[3] * r};
      subtract_viscous_flux(uvL, qL, r, v3, ph.gamma, ph.mu, ph.prandtl, g);   // g = -fv(uL)
#pragma unroll
      for (int k = 0; k < 5; ++k) F[k] += wL * (g[0][k] * n[0] + g[1][k] * n[1] + g[2][k] * n[2]);
    }
    if (wR != T(0)) {
#pragma unroll
      for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int k = 0; k < 5; ++k) g[i][k] = T(0);
      const T r = T(1) / uvR[0];
      const T v3[3] = {uvR[1] * r, uvR[2] * r, uvR[3] * r};
      subtract_viscous_flux(uvR, qR, r, v3, ph.gamma, ph.mu, ph.prandtl, g);
#pragma unroll
      for (int k = 0; k < 5; ++k) F[k] += wR * (g[0][k] * n[0] + g[1][k] * n[1] + g[2][k] * n[2]);
    }
#pragma unroll
    for (int k = 0; k < 5; ++k) F[k] += ph.tau * (uL[k] - pen[k]);
  }
}

// No-slip isothermal wall (reading R11): ghost state for the Riemann problem and wall state.
template <typename T>
__device__ __forceinline__ void ghost_wall(const T uL[5], T e_w, T ub[5], T uw[5]) {
  const T ke = T(0.5) * (uL[1] * uL[1] + uL[2] * uL[2] + uL[3] * uL[3]) / uL[0];
  ub[0] = uL[0];
  ub[1] = -uL[1];
  ub[2] = -uL[2];
  ub[3] = -uL[3];
  ub[4] = uL[0] * e_w + ke;
  uw[0] = uL[0];
  uw[1] = uw[2] = uw[3] = T(0);
  uw[4] = uL[0] * e_w;
}

// Riemann-invariant far field (reading R11).  par = rho_inf, v_inf[3], p_inf.
template <typename T>
__device__ __forceinline__ void ghost_farfield(const T uL[5], const T n[3], T gamma, const T par[5], T ub[5]) {
  const T g1 = gamma - T(1);
  const T rho = uL[0], rr = T(1) / rho;
  const T v[3] = {uL[1] * rr, uL[2] * rr, uL[3] * rr};
  const T p = g1 * (uL[4] - T(0.5) * rho * (v[0] * v[0] + v[1] * v[1] + v[2] * v[2]));
  const T c = fr_sqrt(gamma * p * rr);
  const T vn = v[0] * n[0] + v[1] * n[1] + v[2] * n[2];
  const T rho_i = par[0], p_i = par[4];
  const T c_i = fr_sqrt(gamma * p_i / rho_i);
  const T vn_i = par[1] * n[0] + par[2] * n[1] + par[3] * n[2];
  const T Rp = (vn_i <= -c_i) ? vn_i + T(2) * c_i / g1 : vn + T(2) * c / g1;
  const T Rm = (vn >= c) ? vn - T(2) * c / g1 : vn_i - T(2) * c_i / g1;
  const T vnb = T(0.5) * (Rp + Rm);
  const T cb = T(0.25) * g1 * (Rp - Rm);
  const bool inflow = vnb < T(0);
  const T s_b = inflow ? p_i / pow(rho_i, gamma) : p / pow(rho, gamma);
  T vb[3];
#pragma unroll
  for (int i = 0; i < 3; ++i) vb[i] = inflow ? par[1 + i] + (vnb - vn_i) * n[i] : v[i] + (vnb - vn) * n[i];
  const T rho_b = pow(cb * cb / (gamma * s_b), T(1) / g1);
  const T p_b = rho_b * cb * cb / gamma;
  ub[0] = rho_b;
  ub[1] = rho_b * vb[0];
  ub[2] = rho_b * vb[1];
  ub[3] = rho_b * vb[2];
  ub[4] = p_b / g1 + T(0.5) * rho_b * (vb[0] * vb[0] + vb[1] * vb[1] + vb[2] * vb[2]);
}

}  // namespace frb
