// Element-per-thread fused kernels for small dense elements (fr_element.cu): launch entry points used by the generic driver.
#pragma once
#include "fr_dev.hpp"

namespace fr {

bool element_fused_supported(const DevConsts &c);

// U^f = M0 U -> uf [Nf][NV][ld]
cudaError_t element_interp(const DevConsts &c, const void *u, double *uf, cudaStream_t s);

// Q = J^-T {(M4 - M6 M0) U + M6 C} -> q [nd][Nu][NV][ld];  G^f = n . f_vis(U^f, M0 Q) -> gf [Nf][NV][ld]
cudaError_t element_gradface(const DevConsts &c, const void *u, const double *cf, const double *uf, double *q, double *gf, cudaStream_t s);

// rhs = -(1/J) {(M1 - M3 M2) S f(U, Q) + M3 D~}
cudaError_t element_fluxdiv(const DevConsts &c, const void *u, const double *q, const double *dt, void *rhs, cudaStream_t s);

}  // namespace fr
