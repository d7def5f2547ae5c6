// Generic FR right-hand side: the paper's staged kernel sequence (App A) with dense
// operator matrices, for any element type (FR_FLAG_FORCE_GENERIC; triangles with p = 0 or p > 4; hexahedra with p = 0 or
// p > 6), and the interface (flux-point pair) kernels every path shares.  Triangles and quadrilaterals with 1 <= p <= 4 run
// the fused kernels of fr_element.cu, quadrilaterals of other orders the line kernels of fr_tensor.cu, hexahedra with
// 1 <= p <= 6 the TMA kernels.  All arithmetic in double; u / rhs are stored in T (float or double).
#include "fr_dev.hpp"
#include "fr_element.hpp"
#include "fr_hex_tma.hpp"

namespace fr {
namespace {

constexpr int RT = 8;  // rows of the operator per thread
constexpr int FLUXG_MINB = 6;  // resident CTAs of the gather-bound interface kernels: occupancy is what hides their latency

// out[blk][r][col] = sum_k A[r][k] in1[blk][k][col] (+ sum_k B[r][k] in2[k][col]),  col = a*ld + e.
// SCALE: multiply by -rcpj[r][e] (Eq 19 :243, the paper's negdivconf kernel).
template <typename TIN, typename TOUT, bool SCALE>
__global__ void __launch_bounds__(128) k_apply(int M, int K1, const double *__restrict__ A, const TIN *__restrict__ in1, int K2,
                                               const double *__restrict__ B, const double *__restrict__ in2, TOUT *__restrict__ out,
                                               int64_t ld, int64_t Nel, int NV, const double *__restrict__ rcpj,
                                               int64_t in_blk, int64_t out_blk) {
  extern __shared__ double sA[];  // [RT][K1] then [RT][K2]
  const int r0 = blockIdx.y * RT;
  const int nr = min(RT, M - r0);
  for (int i = threadIdx.x; i < RT * K1; i += blockDim.x) { int j = i / K1, k = i % K1; sA[i] = j < nr ? A[(size_t)(r0 + j) * K1 + k] : 0.0; }
  double *sB = sA + RT * K1;
  for (int i = threadIdx.x; i < RT * K2; i += blockDim.x) { int j = i / K2, k = i % K2; sB[i] = j < nr ? B[(size_t)(r0 + j) * K2 + k] : 0.0; }
  __syncthreads();
  const int64_t ncols = (int64_t)NV * ld;
  const int64_t col = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (col >= ncols) return;
  const int64_t e = col % ld;
  if (e >= Nel) return;
  in1 += (size_t)blockIdx.z * in_blk;
  out += (size_t)blockIdx.z * out_blk;
  double acc[RT];
#pragma unroll
  for (int j = 0; j < RT; ++j) acc[j] = 0.0;
  for (int k = 0; k < K1; ++k) {
    const double x = (double)in1[(size_t)k * ncols + col];
#pragma unroll
    for (int j = 0; j < RT; ++j) acc[j] = fma(sA[j * K1 + k], x, acc[j]);
  }
  for (int k = 0; k < K2; ++k) {
    const double x = in2[(size_t)k * ncols + col];
#pragma unroll
    for (int j = 0; j < RT; ++j) acc[j] = fma(sB[j * K2 + k], x, acc[j]);
  }
#pragma unroll
  for (int j = 0; j < RT; ++j)
    if (j < nr) {
      double v = acc[j];
      if (SCALE) v = -v * rcpj[(size_t)(r0 + j) * ld + e];
      out[(size_t)(r0 + j) * ncols + col] = (TOUT)v;
    }
}

// Common solution, Eq 7 + Eq 25 (:192, :506): each pair visited once, same value to both sides.  Flux-point states and the
// output are in the perturbation variables w (fr_physics.cuh): the gradient kernels differentiate w.
template <int ND, bool JUMP>
__global__ void k_common_sol(DevConsts c, const double *__restrict__ uf, double *__restrict__ cf) {
  constexpr int NV = ND + 2;
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= c.npairs) return;
  const size_t oL = fp_row(c.blk, c.ld, c.Nf * NV, c.pLs[i] * NV, c.pLe[i]), oR = fp_row(c.blk, c.ld, c.Nf * NV, c.pRs[i] * NV, c.pRe[i]);
  const size_t vs = fp_rstride(c.blk, c.ld);  // distance between the variables of one flux point
  const double wl = 0.5 - c.ph.beta, wr = 0.5 + c.ph.beta;
#pragma unroll
  for (int a = 0; a < NV; ++a) {
    const double ul = uf[oL + (size_t)a * vs], ur = uf[oR + (size_t)a * vs];
    const double v = wl * ul + wr * ur;
    cf[oL + (size_t)a * vs] = JUMP ? v - ul : v;   // JUMP: the {C - u^f} of Eq 9 directly
    cf[oR + (size_t)a * vs] = JUMP ? v - ur : v;
  }
}

// Boundary common solution C(u_L, B_ldg u_L)  (:797)
template <int ND, bool JUMP>
__global__ void k_common_sol_bnd(DevConsts c, const double *__restrict__ uf, double *__restrict__ cf) {
  constexpr int NV = ND + 2;
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= c.nbnd) return;
  const size_t o = fp_row(c.blk, c.ld, c.Nf * NV, c.bs[i] * NV, c.be[i]);
  const size_t vs = fp_rstride(c.blk, c.ld);
  double w[NV], u[NV], gi[NV], gl[NV];
#pragma unroll
  for (int a = 0; a < NV; ++a) w[a] = uf[o + (size_t)a * vs];
  from_pert<ND>(c.ph, w, u);
  ghost_states<ND>(c.bcs[c.bbc[i]], u, c.ph.gamma, gi, gl);
  to_pert<ND>(c.ph, gl, gl);
#pragma unroll
  for (int a = 0; a < NV; ++a) cf[o + (size_t)a * vs] = (0.5 - c.ph.beta) * w[a] + (0.5 + c.ph.beta) * gl[a] - (JUMP ? w[a] : 0.0);
}

// q = J^-T q~ = (1/J) S^T q~, Eq 10 (:206), in place
template <int ND>
__global__ void k_grad_phys(DevConsts c, double *__restrict__ qu) {
  constexpr int NV = ND + 2;
  const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= (int64_t)c.Nu * c.ld) return;
  const int64_t e = idx % c.ld, r = idx / c.ld;
  if (e >= c.Nel) return;
  double S[ND][ND];
#pragma unroll
  for (int i = 0; i < ND; ++i)
#pragma unroll
    for (int n = 0; n < ND; ++n) S[i][n] = c.smat[((size_t)(i * ND + n) * c.Nu + r) * c.ld + e];
  const double rj = c.rcpj[(size_t)r * c.ld + e];
#pragma unroll
  for (int a = 0; a < NV; ++a) {
    double qt[ND];
#pragma unroll
    for (int i = 0; i < ND; ++i) qt[i] = qu[(((size_t)i * c.Nu + r) * NV + a) * c.ld + e];
#pragma unroll
    for (int n = 0; n < ND; ++n) {
      double s = 0;
#pragma unroll
      for (int i = 0; i < ND; ++i) s = fma(S[i][n], qt[i], s);
      qu[(((size_t)n * c.Nu + r) * NV + a) * c.ld + e] = s * rj;
    }
  }
}

// F~ = S (f_inv - f_vis), Eq 12 (:214) with Eq 20-24; in place over Q^u
template <int ND, bool NS, typename T>
__global__ void k_tflux(DevConsts c, const T *__restrict__ u, double *__restrict__ qu) {
  constexpr int NV = ND + 2;
  const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= (int64_t)c.Nu * c.ld) return;
  const int64_t e = idx % c.ld, r = idx / c.ld;
  if (e >= c.Nel) return;
  double uu[NV], f[ND][NV], v[ND], p;
#pragma unroll
  for (int a = 0; a < NV; ++a) uu[a] = (double)u[((size_t)r * NV + a) * c.ld + e];
  inviscid_flux<ND>(uu, c.ph, f, v, p);  // staged path: no reference state (w = u)
  if (NS) {
    double q[ND][NV];
#pragma unroll
    for (int n = 0; n < ND; ++n)
#pragma unroll
      for (int a = 0; a < NV; ++a) q[n][a] = qu[(((size_t)n * c.Nu + r) * NV + a) * c.ld + e];
    subtract_viscous_flux<ND>(uu, q, v, c.ph, f);
  }
  double S[ND][ND];
#pragma unroll
  for (int i = 0; i < ND; ++i)
#pragma unroll
    for (int n = 0; n < ND; ++n) S[i][n] = c.smat[((size_t)(i * ND + n) * c.Nu + r) * c.ld + e];
#pragma unroll
  for (int i = 0; i < ND; ++i)
#pragma unroll
    for (int a = 0; a < NV; ++a) {
      double s = 0;
#pragma unroll
      for (int n = 0; n < ND; ++n) s = fma(S[i][n], f[n][a], s);
      qu[(((size_t)i * c.Nu + r) * NV + a) * c.ld + e] = s;
    }
}

// unit normal of the L side and J n of both sides of pair i (Eq 14-16): per-pair tables in iteration order, or the per-face
// tables of an affine hexahedral mesh (fr_dev.hpp: pf_n)
template <int ND, typename TI>
__device__ __forceinline__ void pair_normals(const DevConsts &c, int64_t i, double *nrm, double &jl, double &jr) {
  if (c.pf_n) {
    const int fL = c.pLs[i] / c.nfp, fR = c.pRs[i] / c.nfp;
    const size_t eL = (size_t)c.pLe[i], eR = (size_t)c.pRe[i];
#pragma unroll
    for (int n = 0; n < ND; ++n) nrm[n] = (double)((const TI *)c.pf_n)[((size_t)n * 2 * ND + fL) * c.ld + eL];
    jl = (double)((const TI *)c.pf_Jn)[(size_t)fL * c.ld + eL];
    jr = (double)((const TI *)c.pf_Jn)[(size_t)fR * c.ld + eR];
    return;
  }
#pragma unroll
  for (int n = 0; n < ND; ++n) nrm[n] = (double)((const TI *)c.pn)[(size_t)n * c.npairs + i];  // tables in TI (fr_api.cu)
  jl = (double)((const TI *)c.pJnL)[i];
  jr = (double)((const TI *)c.pJnR)[i];
}

// Common normal flux over flux-point pairs, Eq 15-17 (:227-235); in place over U^f -> D~ (:300)
// TI: storage type of the flux-point arrays (double; float on the hexahedral TMA path in single precision)
template <int ND, bool NS, typename TI>
__global__ void __launch_bounds__(128, NS ? 2 : FLUXG_MINB) k_common_flux(DevConsts c, TI *__restrict__ uf, const TI *__restrict__ qf) {
  constexpr int NV = ND + 2;
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= c.npairs) return;
  const size_t oL = fp_row(c.blk, c.ld, c.Nf * NV, c.pLs[i] * NV, c.pLe[i]), oR = fp_row(c.blk, c.ld, c.Nf * NV, c.pRs[i] * NV, c.pRe[i]);
  const size_t vs = fp_rstride(c.blk, c.ld);  // distance between the variables of one flux point
  const size_t blk = (size_t)c.Nf * NV * c.ld;
  double uL[NV], uR[NV], qL[ND][NV], qR[ND][NV], nrm[ND], F[NV];
#pragma unroll
  for (int a = 0; a < NV; ++a) { uL[a] = (double)uf[oL + (size_t)a * vs]; uR[a] = (double)uf[oR + (size_t)a * vs]; }
  if (NS) {
#pragma unroll
    for (int n = 0; n < ND; ++n)
#pragma unroll
      for (int a = 0; a < NV; ++a) { qL[n][a] = (double)qf[n * blk + oL + (size_t)a * vs]; qR[n][a] = (double)qf[n * blk + oR + (size_t)a * vs]; }
  }
  double jl, jr;
  pair_normals<ND, TI>(c, i, nrm, jl, jr);
  common_flux<ND, NS>(uL, uR, uR, qL, qR, nrm, c.ph, F);
#pragma unroll
  for (int a = 0; a < NV; ++a) { uf[oL + (size_t)a * vs] = (TI)(jl * F[a]); uf[oR + (size_t)a * vs] = (TI)(-jr * F[a]); }
}

template <int ND, bool NS, typename TI>
__global__ void k_common_flux_bnd(DevConsts c, TI *__restrict__ uf, const TI *__restrict__ qf) {
  constexpr int NV = ND + 2;
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= c.nbnd) return;
  const size_t o = fp_row(c.blk, c.ld, c.Nf * NV, c.bs[i] * NV, c.be[i]);
  const size_t vs = fp_rstride(c.blk, c.ld);
  const size_t blk = (size_t)c.Nf * NV * c.ld;
  double uL[NV], gi[NV], gl[NV], qL[ND][NV], qR[ND][NV], nrm[ND], F[NV];
#pragma unroll
  for (int a = 0; a < NV; ++a) uL[a] = (double)uf[o + (size_t)a * vs];
  double uc[NV];
  from_pert<ND>(c.ph, uL, uc);
  const double keep = ghost_states<ND>(c.bcs[c.bbc[i]], uc, c.ph.gamma, gi, gl);
  to_pert<ND>(c.ph, gi, gi);
  to_pert<ND>(c.ph, gl, gl);
  if (NS) {
#pragma unroll
    for (int n = 0; n < ND; ++n)
#pragma unroll
      for (int a = 0; a < NV; ++a) { qL[n][a] = (double)qf[n * blk + o + (size_t)a * vs]; qR[n][a] = keep * qL[n][a]; }
  }
#pragma unroll
  for (int n = 0; n < ND; ++n) nrm[n] = c.bn[(size_t)n * c.nbnd + i];  // boundary tables stay double
  common_flux<ND, NS>(uL, gl, gi, qL, qR, nrm, c.ph, F);
  const double jn = c.bJn[i];
#pragma unroll
  for (int a = 0; a < NV; ++a) uf[o + (size_t)a * vs] = (TI)(jn * F[a]);
}

// Common normal flux with the viscous part pre-contracted by the element kernels (fr_hex_tma.cu):
// gf = n_own . f_vis(u^f, q^f) at every flux point with the element's OWN outward normal, so that
// n_L . f_R^vis = -gf_R.   F = Rusanov + tau (u_L - u_R) - {(1/2+beta) gf_L - (1/2-beta) gf_R}   (Eq 26-27, A7)
template <int ND, typename TI>
__global__ void __launch_bounds__(128, FLUXG_MINB) k_common_flux_g(DevConsts c, TI *__restrict__ uf, const TI *__restrict__ gf) {
  constexpr int NV = ND + 2;
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= c.npairs) return;
  const size_t oL = fp_row(c.blk, c.ld, c.Nf * NV, c.pLs[i] * NV, c.pLe[i]), oR = fp_row(c.blk, c.ld, c.Nf * NV, c.pRs[i] * NV, c.pRe[i]);
  const size_t vs = fp_rstride(c.blk, c.ld);  // distance between the variables of one flux point
  const double wl = 0.5 + c.ph.beta, wr = 0.5 - c.ph.beta;
  double uL[NV], uR[NV], gL[NV], gR[NV], nrm[ND], F[NV];
#pragma unroll
  for (int a = 0; a < NV; ++a) { uL[a] = (double)uf[oL + (size_t)a * vs]; uR[a] = (double)uf[oR + (size_t)a * vs]; }
#pragma unroll
  for (int a = 0; a < NV; ++a) { gL[a] = wl != 0.0 ? (double)gf[oL + (size_t)a * vs] : 0.0; gR[a] = wr != 0.0 ? (double)gf[oR + (size_t)a * vs] : 0.0; }
  double jl, jr;
  pair_normals<ND, TI>(c, i, nrm, jl, jr);
  rusanov<ND>(uL, uR, nrm, c.ph, F);
#pragma unroll
  for (int a = 0; a < NV; ++a) {
    const double f = F[a] + c.ph.tau * (uL[a] - uR[a]) - (wl * gL[a] - wr * gR[a]);
    uf[oL + (size_t)a * vs] = (TI)(jl * f);
    uf[oR + (size_t)a * vs] = (TI)(-jr * f);
  }
}

// boundary flux points: gf already holds the complete LDG viscous flux with the ghost state (App C)
template <int ND, typename TI>
__global__ void k_common_flux_bnd_g(DevConsts c, TI *__restrict__ uf, const TI *__restrict__ gf) {
  constexpr int NV = ND + 2;
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= c.nbnd) return;
  const size_t o = fp_row(c.blk, c.ld, c.Nf * NV, c.bs[i] * NV, c.be[i]);
  const size_t vs = fp_rstride(c.blk, c.ld);
  double uL[NV], gi[NV], gl[NV], nrm[ND], F[NV];
#pragma unroll
  for (int a = 0; a < NV; ++a) uL[a] = (double)uf[o + (size_t)a * vs];
  double uc[NV];
  from_pert<ND>(c.ph, uL, uc);
  ghost_states<ND>(c.bcs[c.bbc[i]], uc, c.ph.gamma, gi, gl);
  to_pert<ND>(c.ph, gi, gi);
  to_pert<ND>(c.ph, gl, gl);
#pragma unroll
  for (int n = 0; n < ND; ++n) nrm[n] = c.bn[(size_t)n * c.nbnd + i];
  rusanov<ND>(uL, gi, nrm, c.ph, F);
  const double jn = c.bJn[i];
#pragma unroll
  for (int a = 0; a < NV; ++a) uf[o + (size_t)a * vs] = (TI)(jn * (F[a] + c.ph.tau * (uL[a] - gl[a]) - (double)gf[o + (size_t)a * vs]));
}

template <typename TIN, typename TOUT, bool SCALE>
void apply(cudaStream_t s, const DevConsts &c, int M, int K1, const double *A, const TIN *in1, int K2, const double *B,
           const double *in2, TOUT *out, int nblk = 1, int64_t in_blk = 0, int64_t out_blk = 0) {
  const int64_t ncols = (int64_t)c.NV * c.ld;
  dim3 grid((unsigned)((ncols + 127) / 128), (unsigned)((M + RT - 1) / RT), (unsigned)nblk);
  size_t smem = (size_t)RT * (K1 + K2) * sizeof(double);
  if (smem > 48 * 1024) cudaFuncSetAttribute(k_apply<TIN, TOUT, SCALE>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  k_apply<TIN, TOUT, SCALE><<<grid, 128, smem, s>>>(M, K1, A, in1, K2, B, in2, out, c.ld, c.Nel, c.NV, c.rcpj, in_blk, out_blk);
}

template <int ND, bool NS, typename T>
cudaError_t run(const DevConsts &c, const WorkLayout &w, const T *u, T *rhs, char *work, cudaStream_t s, Prof *prof) {
  double *uf = (double *)(work + w.uf), *cf = (double *)(work + w.cf), *qu = (double *)(work + w.qu), *qf = (double *)(work + w.qf);
  const int Nu = c.Nu, Nf = c.Nf;
  const int TB = 128;
  auto blocks = [&](int64_t n) { return (unsigned)((n + TB - 1) / TB); };
  const int64_t npts = (int64_t)Nu * c.ld;
  if (ND == 2 && element_fused_supported(c)) {
    // triangles: fused kernels with one thread per (element, variable) (fr_element.cu), 5 launches (3 for Euler);
    // Q^f and F~ are never stored
    FR_MARK(prof, "el_interp");
    cudaError_t e = element_interp(c, u, uf, s);
    if (e != cudaSuccess) return e;
    if (NS) {
      // the gradient kernel forms the common solution of interior flux points itself (c.fp_poff); boundaries keep their kernel
      FR_MARK(prof, "el_gradface");
      if (!c.fp_poff && c.npairs) k_common_sol<ND, false><<<blocks(c.npairs), TB, 0, s>>>(c, uf, cf);
      if (c.nbnd) k_common_sol_bnd<ND, false><<<blocks(c.nbnd), TB, 0, s>>>(c, uf, cf);
      if ((e = element_gradface(c, u, cf, uf, qu, qf, s)) != cudaSuccess) return e;
      FR_MARK(prof, "common_flux_g");
      launch_common_flux_g(c, uf, qf, false, s);
    } else {
      FR_MARK(prof, "common_flux");
      if (c.npairs) k_common_flux<ND, NS, double><<<blocks(c.npairs), TB, 0, s>>>(c, uf, qf);
      if (c.nbnd) k_common_flux_bnd<ND, NS, double><<<blocks(c.nbnd), TB, 0, s>>>(c, uf, qf);
    }
    FR_MARK(prof, "el_fluxdiv");
    e = element_fluxdiv(c, u, qu, uf, rhs, s);
    return e != cudaSuccess ? e : cudaGetLastError();
  }
  // (1) U^f = M0 U                                                       Eq 41 :745
  FR_MARK(prof, "apply_M0");
  apply<T, double, false>(s, c, Nf, Nu, c.M0, u, 0, nullptr, nullptr, uf);
  if (NS) {
    // (2) C^f                                                            Eq 7, 25
    FR_MARK(prof, "common_sol");
    if (c.npairs) k_common_sol<ND, false><<<blocks(c.npairs), TB, 0, s>>>(c, uf, cf);
    if (c.nbnd) k_common_sol_bnd<ND, false><<<blocks(c.nbnd), TB, 0, s>>>(c, uf, cf);
    // (2) Q~ = (M4 - M6 M0) U + M6 C                                     Eq 42 :756
    FR_MARK(prof, "apply_M46_M6");
    apply<T, double, false>(s, c, ND * Nu, Nu, c.M46, u, Nf, c.M6, cf, qu);
    // (3) Q = J^-T Q~ ; Q^f = M5 Q                                       Eq 10, Eq 43
    FR_MARK(prof, "grad_phys");
    k_grad_phys<ND><<<blocks(npts), TB, 0, s>>>(c, qu);
    FR_MARK(prof, "apply_M5");
    apply<double, double, false>(s, c, Nf, Nu, c.M0, qu, 0, nullptr, nullptr, qf, ND, (int64_t)Nu * c.NV * c.ld, (int64_t)Nf * c.NV * c.ld);
  }
  // (4) F~ = S f(U, Q)                                                   Eq 12
  FR_MARK(prof, "tflux");
  k_tflux<ND, NS, T><<<blocks(npts), TB, 0, s>>>(c, u, qu);
  // (5) D~ = J n F(...)  in place over U^f                               Eq 15-17
  FR_MARK(prof, "common_flux");
  if (c.npairs) k_common_flux<ND, NS, double><<<blocks(c.npairs), TB, 0, s>>>(c, uf, qf);
  if (c.nbnd) k_common_flux_bnd<ND, NS, double><<<blocks(c.nbnd), TB, 0, s>>>(c, uf, qf);
  // (6,7) R = -(1/J) {(M1 - M3 M2) F~ + M3 D~}                           Eq 44, Eq 19
  FR_MARK(prof, "apply_M132_M3_negdivconf");
  apply<double, T, true>(s, c, Nu, ND * Nu, c.M132, qu, Nf, c.M3, uf, rhs);
  return cudaGetLastError();
}

}  // namespace

// launchers shared with the tensor-product path (fr_tensor.cu)
void launch_common_jump(const DevConsts &c, const double *uf, double *cf, cudaStream_t s) {
  const int TB = 128;
  if (c.nd == 2) {
    if (c.npairs) k_common_sol<2, true><<<(unsigned)((c.npairs + TB - 1) / TB), TB, 0, s>>>(c, uf, cf);
    if (c.nbnd) k_common_sol_bnd<2, true><<<(unsigned)((c.nbnd + TB - 1) / TB), TB, 0, s>>>(c, uf, cf);
  } else {
    if (c.npairs) k_common_sol<3, true><<<(unsigned)((c.npairs + TB - 1) / TB), TB, 0, s>>>(c, uf, cf);
    if (c.nbnd) k_common_sol_bnd<3, true><<<(unsigned)((c.nbnd + TB - 1) / TB), TB, 0, s>>>(c, uf, cf);
  }
}

void launch_common_sol(const DevConsts &c, const double *uf, double *cf, cudaStream_t s) {  // 2-D, C itself (Eq 7)
  const int TB = 128;
  if (c.npairs) k_common_sol<2, false><<<(unsigned)((c.npairs + TB - 1) / TB), TB, 0, s>>>(c, uf, cf);
  if (c.nbnd) k_common_sol_bnd<2, false><<<(unsigned)((c.nbnd + TB - 1) / TB), TB, 0, s>>>(c, uf, cf);
}

template <int ND, bool NS>
static void launch_tflux_t(const DevConsts &c, const void *u, double *qu, cudaStream_t s) {
  const int TB = 128;
  const int64_t npts = (int64_t)c.Nu * c.ld;
  if (c.f64) k_tflux<ND, NS, double><<<(unsigned)((npts + TB - 1) / TB), TB, 0, s>>>(c, (const double *)u, qu);
  else k_tflux<ND, NS, float><<<(unsigned)((npts + TB - 1) / TB), TB, 0, s>>>(c, (const float *)u, qu);
}

void launch_tflux(const DevConsts &c, const void *u, double *qu, cudaStream_t s) {
  if (c.nd == 2) { if (c.ns) launch_tflux_t<2, true>(c, u, qu, s); else launch_tflux_t<2, false>(c, u, qu, s); }
  else { if (c.ns) launch_tflux_t<3, true>(c, u, qu, s); else launch_tflux_t<3, false>(c, u, qu, s); }
}

template <int ND, bool NS, typename TI>
static void launch_common_flux_t(const DevConsts &c, void *uf, const void *qf, cudaStream_t s) {
  const int TB = 128;
  if (c.npairs) k_common_flux<ND, NS, TI><<<(unsigned)((c.npairs + TB - 1) / TB), TB, 0, s>>>(c, (TI *)uf, (const TI *)qf);
  if (c.nbnd) k_common_flux_bnd<ND, NS, TI><<<(unsigned)((c.nbnd + TB - 1) / TB), TB, 0, s>>>(c, (TI *)uf, (const TI *)qf);
}

void launch_common_flux(const DevConsts &c, void *uf, const void *qf, bool f32, cudaStream_t s) {
  if (f32) {  // Euler on the hexahedral TMA path in single precision
    if (c.nd == 3 && !c.ns) launch_common_flux_t<3, false, float>(c, uf, qf, s);
    return;
  }
  if (c.nd == 2) { if (c.ns) launch_common_flux_t<2, true, double>(c, uf, qf, s); else launch_common_flux_t<2, false, double>(c, uf, qf, s); }
  else { if (c.ns) launch_common_flux_t<3, true, double>(c, uf, qf, s); else launch_common_flux_t<3, false, double>(c, uf, qf, s); }
}

template <int ND, typename TI>
static void launch_common_flux_g_t(const DevConsts &c, void *uf, const void *gf, cudaStream_t s) {
  const int TB = 128;
  if (c.npairs) k_common_flux_g<ND, TI><<<(unsigned)((c.npairs + TB - 1) / TB), TB, 0, s>>>(c, (TI *)uf, (const TI *)gf);
  if (c.nbnd) k_common_flux_bnd_g<ND, TI><<<(unsigned)((c.nbnd + TB - 1) / TB), TB, 0, s>>>(c, (TI *)uf, (const TI *)gf);
}

void launch_common_flux_g(const DevConsts &c, void *uf, const void *gf, bool f32, cudaStream_t s) {
  if (c.nd == 2) launch_common_flux_g_t<2, double>(c, uf, gf, s);
  else if (f32) launch_common_flux_g_t<3, float>(c, uf, gf, s);
  else launch_common_flux_g_t<3, double>(c, uf, gf, s);
}

int generic_rhs_launches(const DevConsts &c) {
  if (c.nd == 2 && element_fused_supported(c)) {
    int n = c.ns ? 4 : 3;  // interp, (gradface with the common solution,) common flux, fluxdiv
    if (c.nbnd) n += c.ns ? 2 : 1;
    if (!c.npairs) n -= 1;
    return n;
  }
  int n = 4;  // interp, tflux, common flux, divergence
  if (c.ns) n += 4;  // common solution, gradient, transform, interp of gradient
  if (c.nbnd) n += c.ns ? 2 : 1;
  if (!c.npairs) n -= c.ns ? 2 : 1;
  return n;
}

cudaError_t generic_rhs(const DevConsts &c, const WorkLayout &w, const void *u, void *rhs, char *work, cudaStream_t s, Prof *prof) {
#define FR_RUN(ND, NS)                                                                              \
  (c.f64 ? run<ND, NS, double>(c, w, (const double *)u, (double *)rhs, work, s, prof)                      \
         : run<ND, NS, float>(c, w, (const float *)u, (float *)rhs, work, s, prof))
  if (c.nd == 2) return c.ns ? FR_RUN(2, true) : FR_RUN(2, false);
  return c.ns ? FR_RUN(3, true) : FR_RUN(3, false);
#undef FR_RUN
}

}  // namespace fr
