// TMA-pipelined hexahedral kernels (fr_hex_tma.cu): launch entry points used by the tensor-product driver.
#pragma once
#include "fr_dev.hpp"

namespace fr {

// true when the sm_100a TMA kernels (both of them) can run this n = p+1 / precision: shared memory fits, the driver exposes
// the tensor-map encoder.  The internal arrays are then element-blocked (fr_dev.hpp: fp_row).
bool hex_tma_supported(int n, bool f64);
// cache of encoded tensor maps (one per context; keyed on the u / workspace pointers of a call, which rarely change)
void *hex_tma_cache_create();
void hex_tma_cache_destroy(void *cache);

// Flux-point arrays of this path (U^f -> D~, G^f) and Q are stored in the context's storage precision (double | float),
// element-blocked; all arithmetic is double.
// U^f = M0 U in perturbation variables (part 1; fr_hex_interp_tma.cu)
cudaError_t hex_tma_interp(const DevConsts &c, const double *h_ops, const void *u, void *uf, cudaStream_t s);

// G^f = n . f_vis(U^f, Q^f) at the flux points that carry an LDG weight; Q = J^-T {M4 U + M6 (C - U^f)} with the jump formed
// from the partner's U^f gathered in the kernel (parts 2, 3 of the north_star); Q stored slice-major [N][3][NFP][NV][ld]
cudaError_t hex_tma_gradface(const DevConsts &c, const double *h_ops, const void *u, const void *uf, void *gf, void *q, cudaStream_t s);

// rhs = -(1/J) {(M1 - M3 M2) S f(U, Q) + M3 D~} with Q read back (fr_hex_fluxdiv_tma.cu); Euler: q unused
cudaError_t hex_tma_fluxdiv(const DevConsts &c, const double *h_ops, const void *u, const void *q, const void *dt, void *rhs, cudaStream_t s);
bool hex_tma_fluxdiv_supported(int n, bool f64);

// Eq 15-17 over flux-point pairs with the viscous part taken from G^f; in place over U^f -> D~ (fr_generic.cu).
// f32: the flux-point arrays hold floats (hexahedral TMA path in single precision)
void launch_common_flux_g(const DevConsts &c, void *uf, const void *gf, bool f32, cudaStream_t s);

}  // namespace fr
