// Point-wise physics of the FR right-hand side as device functions (double arithmetic):
// Euler flux Eq 20-21, viscous flux Eq 22-24 (:489-500), Rusanov Eq 45-46
// (:785-789), LDG common flux Eq 26-27 (:510-514), ghost states App C (:799-825).
#pragma once
#include <cuda_runtime.h>

#include "../../include/fr.h"

namespace fr {

struct Phys {
  double gamma, mu, Pr, beta, tau;
};

struct BcDev {
  int kind;
  double rho, v[3], p, cpTw;
};

// f_inv[n][a] of Eq 20 for state u[NV]; also returns pressure and velocities
template <int ND>
__device__ __forceinline__ void inviscid_flux(const double *u, double gamma, double (*f)[ND + 2], double *v, double &p) {
  const double rrho = 1.0 / u[0];
  double ke = 0;
#pragma unroll
  for (int d = 0; d < ND; ++d) { v[d] = u[1 + d] * rrho; ke += u[1 + d] * v[d]; }
  const double E = u[ND + 1];
  p = (gamma - 1.0) * (E - 0.5 * ke);
#pragma unroll
  for (int n = 0; n < ND; ++n) {
    f[n][0] = u[1 + n];
#pragma unroll
    for (int j = 0; j < ND; ++j) f[n][1 + j] = u[1 + n] * v[j] + (j == n ? p : 0.0);
    f[n][ND + 1] = v[n] * (E + p);
  }
}

// f_vis[n][a] of Eq 22-24 SUBTRACTED from f (f -= f_vis).  q[n][a] = d_n u_a.
// d_i v_j by the quotient rule; Delta*dT = (mu*gamma/Pr) d e (A8); 2/3 kept in 2-D (A22).
template <int ND>
__device__ __forceinline__ void subtract_viscous_flux(const double *u, const double (*q)[ND + 2], const double *v,
                                                      const Phys &ph, double (*f)[ND + 2]) {
  const double rrho = 1.0 / u[0];
  const double E = u[ND + 1];
  double dv[ND][ND];
  double div = 0;
#pragma unroll
  for (int i = 0; i < ND; ++i) {
#pragma unroll
    for (int j = 0; j < ND; ++j) dv[i][j] = (q[i][1 + j] - v[j] * q[i][0]) * rrho;
    div += dv[i][i];
  }
  const double lam = -2.0 / 3.0 * ph.mu * div;
  double T[ND][ND];
#pragma unroll
  for (int i = 0; i < ND; ++i)
#pragma unroll
    for (int j = 0; j < ND; ++j) T[i][j] = ph.mu * (dv[i][j] + dv[j][i]) + (i == j ? lam : 0.0);
  const double kap = ph.mu * ph.gamma / ph.Pr;
#pragma unroll
  for (int n = 0; n < ND; ++n) {
    double de = (q[n][ND + 1] - (E * rrho) * q[n][0]) * rrho;
    double vt = 0;
#pragma unroll
    for (int j = 0; j < ND; ++j) { de -= v[j] * dv[n][j]; vt += v[j] * T[j][n]; }
#pragma unroll
    for (int j = 0; j < ND; ++j) f[n][1 + j] -= T[n][j];
    f[n][ND + 1] -= vt + kap * de;
  }
}

// normal viscous flux n . f_vis(u, q)   (used by the LDG interface flux)
template <int ND>
__device__ __forceinline__ void normal_viscous_flux(const double *u, const double (*q)[ND + 2], const double *nrm,
                                                    const Phys &ph, double *fn) {
  double f[ND][ND + 2], v[ND];
  const double rrho = 1.0 / u[0];
#pragma unroll
  for (int d = 0; d < ND; ++d) v[d] = u[1 + d] * rrho;
#pragma unroll
  for (int n = 0; n < ND; ++n)
#pragma unroll
    for (int a = 0; a < ND + 2; ++a) f[n][a] = 0.0;
  subtract_viscous_flux<ND>(u, q, v, ph, f);
#pragma unroll
  for (int a = 0; a < ND + 2; ++a) {
    double s = 0;
#pragma unroll
    for (int n = 0; n < ND; ++n) s -= nrm[n] * f[n][a];
    fn[a] = s;
  }
}

// n . f_inv(u) of Eq 20 contracted with the unit normal directly (5 values instead of the 15 of the flux tensor):
// [rho vn, rho v_j vn + p n_j, (E + p) vn] with vn = n . v; also returns vn and the pressure
template <int ND>
__device__ __forceinline__ void normal_inviscid_flux(const double *u, const double *nrm, double gamma, double *fn, double &vn, double &p) {
  const double rrho = 1.0 / u[0];
  double ke = 0, mn = 0;
#pragma unroll
  for (int d = 0; d < ND; ++d) { ke += u[1 + d] * (u[1 + d] * rrho); mn += nrm[d] * u[1 + d]; }
  const double E = u[ND + 1];
  p = (gamma - 1.0) * (E - 0.5 * ke);
  vn = mn * rrho;
  fn[0] = mn;
#pragma unroll
  for (int j = 0; j < ND; ++j) fn[1 + j] = fma(u[1 + j], vn, p * nrm[j]);
  fn[ND + 1] = vn * (E + p);
}

// Rusanov, Eq 45-46 with the printed wave-speed estimate (A14)
template <int ND>
__device__ __forceinline__ void rusanov(const double *uL, const double *uR, const double *nrm, double gamma, double *F) {
  double fL[ND + 2], fR[ND + 2], vnL, vnR, pL, pR;
  normal_inviscid_flux<ND>(uL, nrm, gamma, fL, vnL, pL);
  normal_inviscid_flux<ND>(uR, nrm, gamma, fR, vnR, pR);
  const double s = sqrt(gamma * (pL + pR) / (uL[0] + uR[0])) + 0.5 * fabs(vnL + vnR);
#pragma unroll
  for (int a = 0; a < ND + 2; ++a) F[a] = 0.5 * (fL[a] + fR[a]) + 0.5 * s * (uL[a] - uR[a]);
}

// Ghost states of Appendix C.  gi: B_inv u_L, gl: B_ldg u_L; returns the factor of q_L in B_ldg q_L.
template <int ND>
__device__ __forceinline__ double ghost_states(const BcDev &bc, const double *uL, double gamma, double *gi, double *gl) {
  const double rho = uL[0], rrho = 1.0 / uL[0];
  double v[ND];
#pragma unroll
  for (int d = 0; d < ND; ++d) v[d] = uL[1 + d] * rrho;
  if (bc.kind == FR_BC_SUP_INFLOW) {  // Eq 47-48
    double ke = 0;
#pragma unroll
    for (int d = 0; d < ND; ++d) { gi[1 + d] = bc.rho * bc.v[d]; ke += bc.v[d] * bc.v[d]; }
    gi[0] = bc.rho; gi[ND + 1] = bc.p / (gamma - 1.0) + 0.5 * bc.rho * ke;
#pragma unroll
    for (int a = 0; a < ND + 2; ++a) gl[a] = gi[a];
    return 0.0;
  }
  if (bc.kind == FR_BC_SUB_OUTFLOW) {  // Eq 49-50
    double ke = 0;
#pragma unroll
    for (int d = 0; d < ND; ++d) { gi[1 + d] = uL[1 + d]; ke += v[d] * v[d]; }
    gi[0] = rho; gi[ND + 1] = bc.p / (gamma - 1.0) + 0.5 * rho * ke;
#pragma unroll
    for (int a = 0; a < ND + 2; ++a) gl[a] = gi[a];
    return 0.0;
  }
  // no-slip isothermal wall, Eq 51-53
  double ki = 0, kw = 0;
#pragma unroll
  for (int d = 0; d < ND; ++d) {
    const double vi = 2.0 * bc.v[d] - v[d];
    gi[1 + d] = rho * vi; gl[1 + d] = rho * bc.v[d];
    ki += vi * vi; kw += bc.v[d] * bc.v[d];
  }
  gi[0] = rho; gl[0] = rho;
  gi[ND + 1] = rho * (bc.cpTw / gamma + 0.5 * ki);
  gl[ND + 1] = rho * (bc.cpTw / gamma + 0.5 * kw);
  return 1.0;
}

// Common normal flux Eq 26 with the penalty in its dissipative sign (A7):
// F = F_inv(uL, uRinv) - n.{(1/2+beta) f_L^vis + (1/2-beta) f_R^vis} + tau (uL - uR)
template <int ND, bool NS>
__device__ __forceinline__ void common_flux(const double *uL, const double *uR, const double *uRinv, const double (*qL)[ND + 2],
                                            const double (*qR)[ND + 2], const double *nrm, const Phys &ph, double *F) {
  rusanov<ND>(uL, uRinv, nrm, ph.gamma, F);
  if (NS) {
    double fvL[ND + 2], fvR[ND + 2];
    const double wl = 0.5 + ph.beta, wr = 0.5 - ph.beta;
    if (wl != 0.0) normal_viscous_flux<ND>(uL, qL, nrm, ph, fvL);
    if (wr != 0.0) normal_viscous_flux<ND>(uR, qR, nrm, ph, fvR);
#pragma unroll
    for (int a = 0; a < ND + 2; ++a) {
      double fv = 0;
      if (wl != 0.0) fv += wl * fvL[a];
      if (wr != 0.0) fv += wr * fvR[a];
      F[a] += ph.tau * (uL[a] - uR[a]) - fv;
    }
  }
}

}  // namespace fr
