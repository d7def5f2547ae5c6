// Point-wise physics of the FR right-hand side as device functions (double arithmetic):
// Euler flux Eq 20-21, viscous flux Eq 22-24 (:489-500), Rusanov Eq 45-46
// (:785-789), LDG common flux Eq 26-27 (:510-514), ghost states App C (:799-825).
#pragma once
#include <cuda_runtime.h>

#include "../../include/fr.h"

namespace fr {

// Gas constants, LDG parameters and the optional constant reference state (fr.h: fr_disc_desc rho_ref, v_ref, p_ref).
//
// Perturbation form.  With a reference state (rho0, v0, p0), E0 = p0/(gamma-1) + rho0 |v0|^2 / 2,
// h0 = (E0 + p0)/rho0, the fused kernels carry the flux-point states and evaluate the inviscid fluxes in the variables
//     w_rho = rho - rho0,   w_mj = m_j - v0_j rho,   w_E = (E - E0) - h0 (rho - rho0)          (w = T (u - u_ref), T constant)
// whose equations are  d_t w + div g = 0  with  g = T f - const:
//     g_rho,n = w_mn + v0_n w_rho,   g_mj,n = v_n w_mj + p' delta_nj,   g_E,n = v_n (w_E + p'),
//     p' = p - p0 = (gamma-1) {w_E + hs0 w_rho - v0 . w_m - |w_m|^2 / (2 rho)},   hs0 = h0 - |v0|^2/2,   v = v0 + w_m / rho.
// T is linear and constant, so interpolation, jumps, Rusanov dissipation s/2 (w_L - w_R), lifting and divergence commute
// with it; the subtracted constant flux has zero discrete divergence (Eq 18: M1 const = 0, common flux of equal states =
// the flux itself).  The right-hand side returns to conserved variables by R_mj = R_wmj + v0_j R_wrho, R_E = R_wE + h0 R_wrho.
// Every O(p0), O(E0) term is gone from the arithmetic: rounding errors scale with the deviation from the reference state.
// The viscous flux is unchanged (f_vis,rho = 0, so T f_vis = f_vis) and is evaluated from conserved variables.
// All-zero reference: w = u, g = f, p' = p -- the plain formulas of Eq 20-21.
struct Phys {
  double gamma, mu, Pr, beta, tau;
  double rho0, v0[3], p0, E0, h0, hs0;
};

inline Phys make_phys(double gamma, double mu, double Pr, double beta, double tau, double rho0, const double *v0, double p0) {
  Phys ph{};
  ph.gamma = gamma; ph.mu = mu; ph.Pr = Pr; ph.beta = beta; ph.tau = tau;
  if (rho0 > 0.0 && p0 > 0.0) {
    double ke = 0;
    for (int d = 0; d < 3; ++d) { ph.v0[d] = v0[d]; ke += v0[d] * v0[d]; }
    ph.rho0 = rho0; ph.p0 = p0;
    ph.E0 = p0 / (gamma - 1.0) + 0.5 * rho0 * ke;
    ph.h0 = (ph.E0 + p0) / rho0;
    ph.hs0 = ph.h0 - 0.5 * ke;
  }
  return ph;
}

struct BcDev {
  int kind;
  double rho, v[3], p, cpTw;
};

// conserved u -> perturbation variables w (may alias)
template <int ND>
__device__ __forceinline__ void to_pert(const Phys &ph, const double *u, double *w) {
  const double rho = u[0], dr = rho - ph.rho0;
  w[ND + 1] = fma(-ph.h0, dr, u[ND + 1] - ph.E0);
#pragma unroll
  for (int d = 0; d < ND; ++d) w[1 + d] = fma(-ph.v0[d], rho, u[1 + d]);
  w[0] = dr;
}
// w -> conserved u (may alias)
template <int ND>
__device__ __forceinline__ void from_pert(const Phys &ph, const double *w, double *u) {
  const double dr = w[0], rho = dr + ph.rho0;
  u[ND + 1] = fma(ph.h0, dr, w[ND + 1]) + ph.E0;
#pragma unroll
  for (int d = 0; d < ND; ++d) u[1 + d] = fma(ph.v0[d], rho, w[1 + d]);
  u[0] = rho;
}
// a difference (jump, increment) of w -> the same difference of u, in place
template <int ND>
__device__ __forceinline__ void from_pert_delta(const Phys &ph, double *d) {
#pragma unroll
  for (int j = 0; j < ND; ++j) d[1 + j] = fma(ph.v0[j], d[0], d[1 + j]);
  d[ND + 1] = fma(ph.h0, d[0], d[ND + 1]);
}

// g[n][a] (Eq 20 in perturbation form) for the perturbation state w[NV]; also returns the full velocities and p' = p - p0
template <int ND>
__device__ __forceinline__ void inviscid_flux(const double *w, const Phys &ph, double (*g)[ND + 2], double *v, double &pp) {
  const double rrho = 1.0 / (w[0] + ph.rho0);
  double ke = 0, vw = 0;
#pragma unroll
  for (int d = 0; d < ND; ++d) {
    const double dv = w[1 + d] * rrho;
    v[d] = ph.v0[d] + dv;
    ke += w[1 + d] * dv;
    vw += ph.v0[d] * w[1 + d];
  }
  const double wE = w[ND + 1];
  pp = (ph.gamma - 1.0) * (fma(ph.hs0, w[0], wE) - vw - 0.5 * ke);
#pragma unroll
  for (int n = 0; n < ND; ++n) {
    g[n][0] = fma(ph.v0[n], w[0], w[1 + n]);
#pragma unroll
    for (int j = 0; j < ND; ++j) g[n][1 + j] = v[n] * w[1 + j] + (j == n ? pp : 0.0);
    g[n][ND + 1] = v[n] * (wE + pp);
  }
}

// f_vis[n][a] of Eq 22-24 SUBTRACTED from f (f -= f_vis), from the perturbation state w and ITS gradient qw[n][a] = d_n w_a
// (T is constant, so grad w = T grad u; differentiating w instead of u keeps the O(E0) terms out of the second derivatives).
// d_i v_j = (d_i w_mj - dv_j d_i rho) / rho with dv = w_m / rho = v - v0 (quotient rule, Galilean invariant);
// Delta*dT = (mu*gamma/Pr) d e (A8) with  d_i E - (E/rho) d_i rho = d_i w_E - ((w_E - p0)/rho) d_i rho;  2/3 kept in 2-D (A22).
// v: the full velocities.  With no reference state these are the plain formulas in conserved variables.
template <int ND>
__device__ __forceinline__ void subtract_viscous_flux(const double *w, const double (*qw)[ND + 2], const double *v,
                                                      const Phys &ph, double (*f)[ND + 2]) {
  const double rrho = 1.0 / (w[0] + ph.rho0);
  const double Es = (w[ND + 1] - ph.p0) * rrho;
  double dv[ND][ND];
  double div = 0;
#pragma unroll
  for (int i = 0; i < ND; ++i) {
#pragma unroll
    for (int j = 0; j < ND; ++j) dv[i][j] = (qw[i][1 + j] - (w[1 + j] * rrho) * qw[i][0]) * rrho;
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
    double de = (qw[n][ND + 1] - Es * qw[n][0]) * rrho;
    double vt = 0;
#pragma unroll
    for (int j = 0; j < ND; ++j) { de -= v[j] * dv[n][j]; vt += v[j] * T[j][n]; }
#pragma unroll
    for (int j = 0; j < ND; ++j) f[n][1 + j] -= T[n][j];
    f[n][ND + 1] -= vt + kap * de;
  }
}

// normal viscous flux n . f_vis(w, grad w)   (used by the LDG interface flux)
template <int ND>
__device__ __forceinline__ void normal_viscous_flux(const double *w, const double (*qw)[ND + 2], const double *nrm,
                                                    const Phys &ph, double *fn) {
  double f[ND][ND + 2], v[ND];
  const double rrho = 1.0 / (w[0] + ph.rho0);
#pragma unroll
  for (int d = 0; d < ND; ++d) v[d] = ph.v0[d] + w[1 + d] * rrho;
#pragma unroll
  for (int n = 0; n < ND; ++n)
#pragma unroll
    for (int a = 0; a < ND + 2; ++a) f[n][a] = 0.0;
  subtract_viscous_flux<ND>(w, qw, v, ph, f);
#pragma unroll
  for (int a = 0; a < ND + 2; ++a) {
    double s = 0;
#pragma unroll
    for (int n = 0; n < ND; ++n) s -= nrm[n] * f[n][a];
    fn[a] = s;
  }
}

// n . g(w) contracted with the unit normal directly (5 values instead of the 15 of the flux tensor):
// [w_m.n + (v0.n) w_rho,  vn w_mj + p' n_j,  vn (w_E + p')]  with vn = n . v (full velocity); also returns vn, p' and rho
template <int ND>
__device__ __forceinline__ void normal_inviscid_flux(const double *w, const double *nrm, const Phys &ph, double *gn, double &vn, double &pp,
                                                     double &rho) {
  rho = w[0] + ph.rho0;
  const double rrho = 1.0 / rho;
  double ke = 0, vw = 0, wn = 0, v0n = 0;
#pragma unroll
  for (int d = 0; d < ND; ++d) {
    ke += w[1 + d] * (w[1 + d] * rrho);
    vw += ph.v0[d] * w[1 + d];
    wn += nrm[d] * w[1 + d];
    v0n += nrm[d] * ph.v0[d];
  }
  const double wE = w[ND + 1];
  pp = (ph.gamma - 1.0) * (fma(ph.hs0, w[0], wE) - vw - 0.5 * ke);
  vn = fma(wn, rrho, v0n);
  gn[0] = fma(v0n, w[0], wn);
#pragma unroll
  for (int j = 0; j < ND; ++j) gn[1 + j] = fma(w[1 + j], vn, pp * nrm[j]);
  gn[ND + 1] = vn * (wE + pp);
}

// Rusanov, Eq 45-46 with the printed wave-speed estimate (A14), on perturbation states: the dissipation acts on w_L - w_R
template <int ND>
__device__ __forceinline__ void rusanov(const double *wL, const double *wR, const double *nrm, const Phys &ph, double *F) {
  double fL[ND + 2], fR[ND + 2], vnL, vnR, pL, pR, rL, rR;
  normal_inviscid_flux<ND>(wL, nrm, ph, fL, vnL, pL, rL);
  normal_inviscid_flux<ND>(wR, nrm, ph, fR, vnR, pR, rR);
  const double s = sqrt(ph.gamma * (2.0 * ph.p0 + pL + pR) / (rL + rR)) + 0.5 * fabs(vnL + vnR);
#pragma unroll
  for (int a = 0; a < ND + 2; ++a) F[a] = 0.5 * (fL[a] + fR[a]) + 0.5 * s * (wL[a] - wR[a]);
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

// Common normal flux Eq 26 with the penalty in its dissipative sign (A7), on perturbation states w and their gradients
// (the viscous flux has a zero mass row, so it is the same in both sets of variables):
// F = F_inv(wL, wRinv) - n.{(1/2+beta) f_L^vis + (1/2-beta) f_R^vis} + tau (wL - wR)
template <int ND, bool NS>
__device__ __forceinline__ void common_flux(const double *wL, const double *wR, const double *wRinv, const double (*qL)[ND + 2],
                                            const double (*qR)[ND + 2], const double *nrm, const Phys &ph, double *F) {
  rusanov<ND>(wL, wRinv, nrm, ph, F);
  if (NS) {
    double fvL[ND + 2], fvR[ND + 2];
    const double wl = 0.5 + ph.beta, wr = 0.5 - ph.beta;
    if (wl != 0.0) normal_viscous_flux<ND>(wL, qL, nrm, ph, fvL);
    if (wr != 0.0) normal_viscous_flux<ND>(wR, qR, nrm, ph, fvR);
#pragma unroll
    for (int a = 0; a < ND + 2; ++a) {
      double fv = 0;
      if (wl != 0.0) fv += wl * fvL[a];
      if (wr != 0.0) fv += wr * fvR[a];
      F[a] += ph.tau * (wL[a] - wR[a]) - fv;
    }
  }
}

}  // namespace fr
