// Meshes of several element types: the interface kernels over flux-point pairs whose two sides may lie in
// different parts (fr_mixed.cu).  The element-local kernels are those of fr_element.cu, part by part.
#pragma once
#include "fr_dev.hpp"

namespace fr {

// Cross-part pair table (device).  Offsets are in doubles from the start of a flux-point REGION of the workspace, in which
// the parts' [N_f][N_V][ld] arrays follow each other; the regions U^f (-> D~), C^f and G^f have the same internal layout, so
// one offset addresses all three.  vL / vR: distance between the variables of one flux point (the part's ld).
struct MixedPairs {
  int64_t n = 0;
  const int64_t *oL = nullptr, *oR = nullptr;
  const int32_t *vL = nullptr, *vR = nullptr;
  const double *nrm = nullptr;  // [2][n] unit normal of the L side (Eq 14)
  const double *jL = nullptr, *jR = nullptr;  // J n of each side (Eq 16-17)
};

// C = (1/2 - beta) u_L + (1/2 + beta) u_R to both sides (Eq 7, 25), in perturbation variables
void mixed_common_sol(const MixedPairs &p, const Phys &ph, const double *uf, double *cf, cudaStream_t s);
// D~ = +- J n F in place over U^f; Navier-Stokes: viscous part from G^f (as k_common_flux_g), Euler: Rusanov only
void mixed_common_flux(const MixedPairs &p, const Phys &ph, bool ns, double *uf, const double *gf, cudaStream_t s);

}  // namespace fr
