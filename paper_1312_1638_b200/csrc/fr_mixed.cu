// Interface kernels of mixed-element meshes (2-D: quadrilaterals and triangles sharing edges): one thread per
// flux-point pair, each pair visited once (:194); the two sides are addressed through per-pair offsets because they may
// belong to parts with different N_f and leading dimensions.  Physics as in fr_generic.cu (fr_physics.cuh).
#include "fr_mixed.hpp"

namespace fr {
namespace {

constexpr int ND = 2, NV = 4;

__global__ void __launch_bounds__(128) k_mixed_common_sol(MixedPairs p, Phys ph, const double *__restrict__ uf, double *__restrict__ cf) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= p.n) return;
  const size_t oL = (size_t)p.oL[i], oR = (size_t)p.oR[i], vL = (size_t)p.vL[i], vR = (size_t)p.vR[i];
  const double wl = 0.5 - ph.beta, wr = 0.5 + ph.beta;
#pragma unroll
  for (int a = 0; a < NV; ++a) {
    const double v = wl * uf[oL + a * vL] + wr * uf[oR + a * vR];
    cf[oL + a * vL] = v;
    cf[oR + a * vR] = v;
  }
}

template <bool NS>
__global__ void __launch_bounds__(128) k_mixed_common_flux(MixedPairs p, Phys ph, double *__restrict__ uf, const double *__restrict__ gf) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= p.n) return;
  const size_t oL = (size_t)p.oL[i], oR = (size_t)p.oR[i], vL = (size_t)p.vL[i], vR = (size_t)p.vR[i];
  const double wl = 0.5 + ph.beta, wr = 0.5 - ph.beta;
  double uL[NV], uR[NV], nrm[ND], F[NV];
#pragma unroll
  for (int a = 0; a < NV; ++a) { uL[a] = uf[oL + a * vL]; uR[a] = uf[oR + a * vR]; }
#pragma unroll
  for (int n = 0; n < ND; ++n) nrm[n] = p.nrm[(size_t)n * p.n + i];
  rusanov<ND>(uL, uR, nrm, ph, F);
  const double jl = p.jL[i], jr = p.jR[i];
#pragma unroll
  for (int a = 0; a < NV; ++a) {
    double f = F[a];
    if (NS) {
      // gf = n_own . f_vis with each side's OWN outward normal: n_L . f_R^vis = -gf_R  (Eq 26-27, A7)
      const double gL = wl != 0.0 ? gf[oL + a * vL] : 0.0, gR = wr != 0.0 ? gf[oR + a * vR] : 0.0;
      f += ph.tau * (uL[a] - uR[a]) - (wl * gL - wr * gR);
    }
    uf[oL + a * vL] = jl * f;
    uf[oR + a * vR] = -jr * f;
  }
}

}  // namespace

void mixed_common_sol(const MixedPairs &p, const Phys &ph, const double *uf, double *cf, cudaStream_t s) {
  if (p.n) k_mixed_common_sol<<<(unsigned)((p.n + 127) / 128), 128, 0, s>>>(p, ph, uf, cf);
}

void mixed_common_flux(const MixedPairs &p, const Phys &ph, bool ns, double *uf, const double *gf, cudaStream_t s) {
  if (!p.n) return;
  const unsigned g = (unsigned)((p.n + 127) / 128);
  if (ns) k_mixed_common_flux<true><<<g, 128, 0, s>>>(p, ph, uf, gf);
  else k_mixed_common_flux<false><<<g, 128, 0, s>>>(p, ph, uf, gf);
}

}  // namespace fr
