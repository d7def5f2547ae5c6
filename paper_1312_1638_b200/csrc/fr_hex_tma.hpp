// TMA-pipelined hexahedral kernels (fr_hex_tma.cu): launch entry points used by the tensor-product driver.
#pragma once
#include "fr_dev.hpp"

namespace fr {

// true when the sm_100a TMA kernels (both of them) can run this n = p+1 / precision: shared memory fits, the driver exposes
// the tensor-map encoder.  The internal arrays are then element-blocked (fr_dev.hpp: fp_row).
bool hex_tma_supported(int n, bool f64);

// U^f = M0 U, element-blocked output (part 1; fr_hex_interp_tma.cu)
cudaError_t hex_tma_interp(const DevConsts &c, const double *h_ops, const void *u, double *uf, cudaStream_t s);

// G^f = n . f_vis(U^f, Q^f) at every flux point, Q computed from u and jump = C - U^f  (parts 2b, 3 of the north_star);
// q != NULL: Q is also stored, slice-major [N][3][NV][NFP][ld], for hex_tma_fluxdiv
cudaError_t hex_tma_gradface(const DevConsts &c, const double *h_ops, const void *u, const double *jump, double *gf, double *q,
                             cudaStream_t s);

// rhs = -(1/J) {(M1 - M3 M2) S f(U, Q) + M3 D~} with Q read back (fr_hex_fluxdiv_tma.cu); Euler: q unused
cudaError_t hex_tma_fluxdiv(const DevConsts &c, const double *h_ops, const void *u, const double *q, const double *dt, void *rhs,
                            cudaStream_t s);
bool hex_tma_fluxdiv_supported(int n, bool f64);

// Eq 15-17 over flux-point pairs with the viscous part taken from G^f; in place over U^f -> D~ (fr_generic.cu)
void launch_common_flux_g(const DevConsts &c, double *uf, const double *gf, cudaStream_t s);

}  // namespace fr
