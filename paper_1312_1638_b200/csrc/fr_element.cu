// Fused kernels for 2-D elements with small dense operators (triangles p <= 4, quadrilaterals p <= 4; App A
// matrices are 10 x 12 ... 30 x 10 for a p = 3 triangle).  They replace six of the eight launches of the staged generic
// sequence (fr_generic.cu) by three:
//
//   k_el_interp   : U^f = M0 U (Eq 41).
//   k_el_gradface : Q = J^-T {(M4 - M6 M0) U + M6 C} (Eq 42 :756, Eq 10), Q^f = M0 Q (Eq 43), and at once
//                   G^f = n . f_vis(U^f, Q^f) (Eq 22-24) with the element's own outward normal; writes Q and G^f.
//                   Replaces apply_M46_M6, grad_phys, apply_M5 and makes the N_D N_V N_f array Q^f unnecessary.
//   k_el_fluxdiv  : F~ = S f(U, Q) (Eq 12) and R = -(1/J) {(M1 - M3 M2) F~ + M3 D~} (Eq 44, Eq 19).
//                   Replaces tflux and apply_M132_M3; F~ never reaches HBM.
//
// A CTA owns EB = 32 consecutive elements and runs one thread per (element, conserved variable): every global access is
// a 256-byte row segment of consecutive elements; the operators are kernel parameters (constant bank) read as FMA operands
// by fully unrolled loops; the per-variable intermediates live in registers; the steps that couple the variables
// (viscous flux at a flux point, flux at a solution point) are redistributed over the CTA's threads through a
// [value][element] shared-memory scratch after one barrier.
#include "fr_element.hpp"

#include <cstdlib>
#include <cstring>

namespace fr {
namespace {

// Operators as kernel parameters: they live in the constant bank, every loop over them is fully unrolled, and each FMA takes
// its operator entry as a constant operand (no load instruction, no register) -- the operators are the same for all threads.
template <int NU, int NF>
struct OpsGrad {
  double M46[2 * NU * NU];  // [ND*NU][NU]   M4 - M6 M0
  double M6[2 * NU * NF];   // [ND*NU][NF]
  double M0[NF * NU];       // [NF][NU]
};
template <int NU, int NF>
struct OpsDiv {
  double M132[NU * 2 * NU];  // [NU][ND*NU]  M1 - M3 M2
  double M3[NU * NF];        // [NU][NF]
};
template <int NU, int NF>
struct OpsInterp {
  double M0[NF * NU];
};

constexpr int EB = 32;        // elements per CTA
constexpr int NVT = 4;        // variables (2-D): threads per element
constexpr int TPB = EB * NVT;

// G at one flux point, ND-dimensional: interior n . f_vis(u, q); boundary the complete LDG viscous flux with the App C
// ghost state (as face_visc in fr_tma.cuh)
template <int ND, bool BND>
__device__ __forceinline__ void face_visc_nd(const double *uf, const double (*qf)[ND + 2], const double *nrm, const Phys &ph, int pe,
                                             const BcDev *__restrict__ bcs, double *G) {
  constexpr int NV = ND + 2;
  normal_viscous_flux<ND>(uf, qf, nrm, ph, G);  // uf: perturbation state w^f, qf: its gradient
  if (BND && pe < 0) {
    double uc[NV], gi[NV], gl[NV], qg[ND][NV], GR[NV];
    from_pert<ND>(ph, uf, uc);
    const double keep = ghost_states<ND>(bcs[-1 - pe], uc, ph.gamma, gi, gl);
    to_pert<ND>(ph, gl, gl);
#pragma unroll
    for (int n = 0; n < ND; ++n)
#pragma unroll
      for (int a = 0; a < NV; ++a) qg[n][a] = keep * qf[n][a];
    normal_viscous_flux<ND>(gl, qg, nrm, ph, GR);
    const double wl = 0.5 + ph.beta, wr = 0.5 - ph.beta;
#pragma unroll
    for (int a = 0; a < NV; ++a) G[a] = (wl != 0.0 ? wl * G[a] : 0.0) + (wr != 0.0 ? wr * GR[a] : 0.0);
  }
}

// Variable a of the conserved state at the NU points of element e (uu, read from u) -> the same component of the perturbation
// variables: w_rho = rho - rho0, w_mj = m_j - v0_j rho, w_E = (E - E0) - h0 (rho - rho0); the other threads' density rows are
// re-read (L1 hits: the thread of variable 0 has just loaded them)
template <int NU, typename T>
__device__ __forceinline__ void pert_rows(const Phys &ph, int a, const T *__restrict__ u, size_t ld, int64_t e, double *uu) {
  constexpr int NV = 4;
  if (ph.rho0 == 0.0) return;
  const double ka = a == 0 ? 0.0 : (a == NV - 1 ? ph.h0 : ph.v0[a - 1]);
  const double da = a == 0 ? ph.rho0 : (a == NV - 1 ? ph.E0 : 0.0);
#pragma unroll
  for (int r = 0; r < NU; ++r) {
    const double rho = a == 0 ? uu[r] : (double)u[((size_t)r * NV) * ld + e];
    uu[r] = a == NV - 1 ? fma(-ka, rho - ph.rho0, uu[r] - da) : fma(-ka, rho, uu[r] - da);
  }
}

// U^f = M0 U (Eq 41): u [NU][NV][ld] (T) -> uf [NF][NV][ld]
template <int NU, int NF, typename T>
__global__ void __launch_bounds__(TPB) k_el_interp(const __grid_constant__ OpsInterp<NU, NF> op, DevConsts c, const T *__restrict__ u,
                                                    double *__restrict__ uf) {
  constexpr int NV = 4;
  const int tid = threadIdx.x, el = tid % EB, a = tid / EB;
  const int64_t e = (int64_t)blockIdx.x * EB + el;
  if (e >= c.Nel) return;
  const size_t ld = c.ld;
  double uu[NU];
#pragma unroll
  for (int r = 0; r < NU; ++r) uu[r] = (double)u[((size_t)r * NV + a) * ld + e];
  // perturbation variables (fr_physics.cuh) BEFORE the interpolation, so that its rounding error scales with the deviation
  // from the reference state
  pert_rows<NU, T>(c.ph, a, u, ld, e, uu);
#pragma unroll
  for (int s = 0; s < NF; ++s) {
    double acc = 0;
#pragma unroll
    for (int r = 0; r < NU; ++r) acc = fma(op.M0[s * NU + r], uu[r], acc);
    uf[((size_t)s * NV + a) * ld + e] = acc;
  }
}

// u [NU][NV][ld] (T), cf = common solution C [NF][NV][ld], uf = U^f [NF][NV][ld]; out: q [ND][NU][NV][ld], gf [NF][NV][ld]
// GATHER: the common solution C (Eq 7, 25) is formed here from the own and the partner's U^f (c.fp_poff / c.face_code, set up by
// fr_api.cu for single-type meshes); cf then holds C at boundary flux points only (k_common_sol_bnd).  Otherwise (parts of a
// mixed mesh) cf holds C everywhere.
template <int NU, int NF, bool BND, bool GATHER, typename T>
__global__ void __launch_bounds__(TPB) k_el_gradface(const __grid_constant__ OpsGrad<NU, NF> op, DevConsts c, const T *__restrict__ u,
                                                      const double *__restrict__ cf, const double *__restrict__ uf,
                                                      double *__restrict__ q, double *__restrict__ gf) {
  constexpr int ND = 2, NV = 4;
  extern __shared__ double smem[];
  double *sQf = smem;  // [ND][NV][NF][EB]  gradient at the flux points, all variables
  const int tid = threadIdx.x, el = tid % EB, a = tid / EB;
  const int64_t e0 = (int64_t)blockIdx.x * EB, e = e0 + el;
  const size_t ld = c.ld;
  if (e < c.Nel) {
    double uu[NU], cc[NF], qq[ND][NU];
#pragma unroll
    for (int r = 0; r < NU; ++r) uu[r] = (double)u[((size_t)r * NV + a) * ld + e];
    pert_rows<NU, T>(c.ph, a, u, ld, e, uu);  // the gradient is taken of the perturbation variables (fr_physics.cuh)
    if (GATHER) {
      const double wL = 0.5 - c.ph.beta, wR = 0.5 + c.ph.beta;  // C = wL u_L + wR u_R
#pragma unroll
      for (int s = 0; s < NF; ++s) {
        const int code = c.face_code[(size_t)s * ld + e];
        if (BND && code == 3) {
          cc[s] = cf[((size_t)s * NV + a) * ld + e];
        } else {
          const double own = uf[((size_t)s * NV + a) * ld + e], oth = uf[c.fp_poff[(size_t)s * ld + e] + (size_t)a * ld];
          cc[s] = code == 1 ? wL * own + wR * oth : wL * oth + wR * own;
        }
      }
    } else {
#pragma unroll
      for (int s = 0; s < NF; ++s) cc[s] = cf[((size_t)s * NV + a) * ld + e];
    }
    // affine elements: the metric terms of point 0 serve every point (one load instead of N_u)
    double Sa[ND][ND], rja = 0;
    if (c.affine) {
      rja = c.rcpj[e];
#pragma unroll
      for (int d = 0; d < ND; ++d)
#pragma unroll
        for (int n = 0; n < ND; ++n) Sa[d][n] = c.smat[(size_t)(d * ND + n) * NU * ld + e];
    }
#pragma unroll
    for (int r = 0; r < NU; ++r) {
      double qt[ND];
#pragma unroll
      for (int d = 0; d < ND; ++d) {
        double s = 0;
#pragma unroll
        for (int v = 0; v < NU; ++v) s = fma(op.M46[(d * NU + r) * NU + v], uu[v], s);
#pragma unroll
        for (int v = 0; v < NF; ++v) s = fma(op.M6[(d * NU + r) * NF + v], cc[v], s);
        qt[d] = s;
      }
      const double rj = c.affine ? rja : c.rcpj[(size_t)r * ld + e];
#pragma unroll
      for (int n = 0; n < ND; ++n) {
        double s = 0;
#pragma unroll
        for (int d = 0; d < ND; ++d) s = fma(c.affine ? Sa[d][n] : c.smat[((size_t)(d * ND + n) * NU + r) * ld + e], qt[d], s);
        s *= rj;
        q[(((size_t)n * NU + r) * NV + a) * ld + e] = s;
        qq[n][r] = s;
      }
    }
#pragma unroll
    for (int s = 0; s < NF; ++s)
#pragma unroll
      for (int n = 0; n < ND; ++n) {
        double acc = 0;
#pragma unroll
        for (int r = 0; r < NU; ++r) acc = fma(op.M0[s * NU + r], qq[n][r], acc);
        sQf[((n * NV + a) * NF + s) * EB + el] = acc;
      }
  }
  __syncthreads();
  // flux points of the CTA's elements, redistributed over all threads
#pragma unroll
  for (int t = tid; t < NF * EB; t += TPB) {
    const int el2 = t % EB, s = t / EB;
    const int64_t e2 = e0 + el2;
    if (e2 >= c.Nel) continue;
    double us[NV], qf[ND][NV], nrm[ND], G[NV];
#pragma unroll
    for (int b = 0; b < NV; ++b) us[b] = uf[((size_t)s * NV + b) * ld + e2];
#pragma unroll
    for (int n = 0; n < ND; ++n) {
      nrm[n] = c.fp_n[((size_t)n * NF + s) * ld + e2];
#pragma unroll
      for (int b = 0; b < NV; ++b) qf[n][b] = sQf[((n * NV + b) * NF + s) * EB + el2];
    }
    const int pe = BND ? c.fp_pe[(size_t)s * ld + e2] : 0;
    face_visc_nd<ND, BND>(us, qf, nrm, c.ph, pe, c.bcs, G);
#pragma unroll
    for (int b = 0; b < NV; ++b) gf[((size_t)s * NV + b) * ld + e2] = G[b];
  }
}

// u as above, q [ND][NU][NV][ld], dt = D~ [NF][NV][ld]; rhs like u
template <int NU, int NF, bool NS, typename T>
__global__ void __launch_bounds__(TPB) k_el_fluxdiv(const __grid_constant__ OpsDiv<NU, NF> op, DevConsts c, const T *__restrict__ u,
                                                     const double *__restrict__ q, const double *__restrict__ dt, T *__restrict__ rhs) {
  constexpr int ND = 2, NV = 4;
  extern __shared__ double smem[];
  double *sF = smem;  // [ND][NV][NU][EB]
  const int tid = threadIdx.x, el = tid % EB, a = tid / EB;
  const int64_t e0 = (int64_t)blockIdx.x * EB, e = e0 + el;
  const size_t ld = c.ld;
  // F~ = S f(U, Q) at the solution points of the CTA's elements, one (element, point) per thread and pass
#pragma unroll
  for (int t = tid; t < NU * EB; t += TPB) {
    const int el2 = t % EB, r = t / EB;
    const int64_t e2 = e0 + el2;
    if (e2 >= c.Nel) continue;
    double uu[NV], ww[NV], qq[ND][NV], f[ND][NV], v[ND], p;
#pragma unroll
    for (int b = 0; b < NV; ++b) uu[b] = (double)u[((size_t)r * NV + b) * ld + e2];
    to_pert<ND>(c.ph, uu, ww);
    inviscid_flux<ND>(ww, c.ph, f, v, p);
    if (NS) {
#pragma unroll
      for (int n = 0; n < ND; ++n)
#pragma unroll
        for (int b = 0; b < NV; ++b) qq[n][b] = q[(((size_t)n * NU + r) * NV + b) * ld + e2];
      subtract_viscous_flux<ND>(ww, qq, v, c.ph, f);
    }
#pragma unroll
    for (int d = 0; d < ND; ++d) {
      const int rm = c.affine ? 0 : r;  // affine elements: point 0 serves every point
      const double s0 = c.smat[((size_t)(d * ND + 0) * NU + rm) * ld + e2], s1 = c.smat[((size_t)(d * ND + 1) * NU + rm) * ld + e2];
#pragma unroll
      for (int b = 0; b < NV; ++b) sF[((d * NV + b) * NU + r) * EB + el2] = fma(s0, f[0][b], s1 * f[1][b]);
    }
  }
  __syncthreads();
  const bool act = e < c.Nel;
  const int64_t ec = act ? e : c.Nel - 1;  // inactive lanes of the last CTA repeat a valid element (they take part in the barriers)
  double dd[NF];
#pragma unroll
  for (int s = 0; s < NF; ++s) dd[s] = dt[((size_t)s * NV + a) * ld + ec];
  double fa[ND][NU];  // F~ of this variable at all points of the element
#pragma unroll
  for (int d = 0; d < ND; ++d)
#pragma unroll
    for (int v = 0; v < NU; ++v) fa[d][v] = sF[((d * NV + a) * NU + v) * EB + el];
  double acc[NU];
#pragma unroll
  for (int r = 0; r < NU; ++r) {
    double t = 0;
#pragma unroll
    for (int d = 0; d < ND; ++d)
#pragma unroll
      for (int v = 0; v < NU; ++v) t = fma(op.M132[r * ND * NU + d * NU + v], fa[d][v], t);
#pragma unroll
    for (int s = 0; s < NF; ++s) t = fma(op.M3[r * NF + s], dd[s], t);
    acc[r] = t;
  }
  if (c.ph.rho0 != 0.0) {
    // back to conserved variables: R_mj = R_wmj + v0_j R_wrho, R_E = R_wE + h0 R_wrho (the mass row through shared memory)
    __syncthreads();  // every thread has taken its F~ out of sF
    if (a == 0) {
#pragma unroll
      for (int r = 0; r < NU; ++r) sF[r * EB + el] = acc[r];
    }
    __syncthreads();
    const double ka = a == 0 ? 0.0 : (a == NV - 1 ? c.ph.h0 : c.ph.v0[a - 1]);
#pragma unroll
    for (int r = 0; r < NU; ++r) acc[r] = fma(ka, sF[r * EB + el], acc[r]);
  }
  if (!act) return;
#pragma unroll
  for (int r = 0; r < NU; ++r) rhs[((size_t)r * NV + a) * ld + e] = (T)(-acc[r] * c.rcpj[(size_t)(c.affine ? 0 : r) * ld + e]);
}

template <int NU, int NF, typename T>
cudaError_t gradface_t(const DevConsts &c, const void *u, const double *cf, const double *uf, double *q, double *gf, cudaStream_t s) {
  OpsGrad<NU, NF> op;
  std::memcpy(op.M46, c.hM46, sizeof(op.M46));
  std::memcpy(op.M6, c.hM6, sizeof(op.M6));
  std::memcpy(op.M0, c.hM0, sizeof(op.M0));
  const size_t smem = (size_t)(2 * 4 * NF * EB) * sizeof(double);
  const unsigned grid = (unsigned)((c.Nel + EB - 1) / EB);
  static DevFlags done;  // function attributes are per device
  if (!done.test(c.dev) && smem > 48 * 1024) {
    cudaFuncSetAttribute(k_el_gradface<NU, NF, true, true, T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    cudaFuncSetAttribute(k_el_gradface<NU, NF, false, true, T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    cudaFuncSetAttribute(k_el_gradface<NU, NF, true, false, T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    cudaFuncSetAttribute(k_el_gradface<NU, NF, false, false, T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  }
  done.set(c.dev);
  const bool gather = c.fp_poff != nullptr;
  if (gather) {
    if (c.nbnd) k_el_gradface<NU, NF, true, true, T><<<grid, TPB, smem, s>>>(op, c, (const T *)u, cf, uf, q, gf);
    else k_el_gradface<NU, NF, false, true, T><<<grid, TPB, smem, s>>>(op, c, (const T *)u, cf, uf, q, gf);
  } else {
    if (c.nbnd) k_el_gradface<NU, NF, true, false, T><<<grid, TPB, smem, s>>>(op, c, (const T *)u, cf, uf, q, gf);
    else k_el_gradface<NU, NF, false, false, T><<<grid, TPB, smem, s>>>(op, c, (const T *)u, cf, uf, q, gf);
  }
  return cudaGetLastError();
}

template <int NU, int NF, typename T>
cudaError_t fluxdiv_t(const DevConsts &c, const void *u, const double *q, const double *dt, void *rhs, cudaStream_t s) {
  OpsDiv<NU, NF> op;
  std::memcpy(op.M132, c.hM132, sizeof(op.M132));
  std::memcpy(op.M3, c.hM3, sizeof(op.M3));
  const size_t smem = (size_t)(2 * 4 * NU * EB) * sizeof(double);
  const unsigned grid = (unsigned)((c.Nel + EB - 1) / EB);
  static DevFlags done;
  if (!done.test(c.dev) && smem > 48 * 1024) {
    cudaFuncSetAttribute(k_el_fluxdiv<NU, NF, true, T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    cudaFuncSetAttribute(k_el_fluxdiv<NU, NF, false, T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  }
  done.set(c.dev);
  if (c.ns) k_el_fluxdiv<NU, NF, true, T><<<grid, TPB, smem, s>>>(op, c, (const T *)u, q, dt, (T *)rhs);
  else k_el_fluxdiv<NU, NF, false, T><<<grid, TPB, smem, s>>>(op, c, (const T *)u, q, dt, (T *)rhs);
  return cudaGetLastError();
}

template <int NU, int NF, typename T>
cudaError_t interp_t(const DevConsts &c, const void *u, double *uf, cudaStream_t s) {
  OpsInterp<NU, NF> op;
  std::memcpy(op.M0, c.hM0, sizeof(op.M0));
  k_el_interp<NU, NF, T><<<(unsigned)((c.Nel + EB - 1) / EB), TPB, 0, s>>>(op, c, (const T *)u, uf);
  return cudaGetLastError();
}

}  // namespace

// triangles p = 1 .. 5 (N_u = (p+1)(p+2)/2, N_f = 3 (p+1)) and quadrilaterals p = 1 .. 4 (N_u = (p+1)^2, N_f = 4 (p+1)): at these
// sizes the dense operators cost less than the extra launches and HBM round trips of the staged / sum-factorised sequences.
// Quadrilaterals at p = 4 with Navier-Stokes are the exception: the fused gradient kernel needs 254 registers there and the
// sum-factorised line kernels are faster (16.6 against 14.5 GDOF/s on 768^2 elements); Euler at p = 4 stays fused (51 against
// 31 GDOF/s).  Parts of a mixed mesh always take the fused kernels (force_el): the cross-part pair kernels expect their layout.
bool element_fused_supported(const DevConsts &c) {
  if (c.staged) return false;
  if (c.etype == FR_TRI) return c.n >= 2 && c.n <= 6;
  if (c.etype == FR_QUAD) return c.n >= 2 && c.n <= ((c.force_el || !c.ns) ? 5 : 4);
  return false;
}

#define FR_TRI_CASES(CALL)                     \
  if (c.etype == FR_TRI) {                     \
    switch (c.n) {                             \
      case 2: return CALL(3, 6);               \
      case 3: return CALL(6, 9);               \
      case 4: return CALL(10, 12);             \
      case 5: return CALL(15, 15);             \
      case 6: return CALL(21, 18);             \
      default: return cudaErrorNotSupported;   \
    }                                          \
  }                                            \
  switch (c.n) {                               \
    case 2: return CALL(4, 8);                 \
    case 3: return CALL(9, 12);                \
    case 4: return CALL(16, 16);               \
    case 5: return CALL(25, 20);               \
    default: return cudaErrorNotSupported;     \
  }

cudaError_t element_interp(const DevConsts &c, const void *u, double *uf, cudaStream_t s) {
#define FR_CALL(NU, NF) (c.f64 ? interp_t<NU, NF, double>(c, u, uf, s) : interp_t<NU, NF, float>(c, u, uf, s))
  FR_TRI_CASES(FR_CALL)
#undef FR_CALL
}

cudaError_t element_gradface(const DevConsts &c, const void *u, const double *cf, const double *uf, double *q, double *gf, cudaStream_t s) {
#define FR_CALL(NU, NF) (c.f64 ? gradface_t<NU, NF, double>(c, u, cf, uf, q, gf, s) : gradface_t<NU, NF, float>(c, u, cf, uf, q, gf, s))
  FR_TRI_CASES(FR_CALL)
#undef FR_CALL
}

cudaError_t element_fluxdiv(const DevConsts &c, const void *u, const double *q, const double *dt, void *rhs, cudaStream_t s) {
#define FR_CALL(NU, NF) (c.f64 ? fluxdiv_t<NU, NF, double>(c, u, q, dt, rhs, s) : fluxdiv_t<NU, NF, float>(c, u, q, dt, rhs, s))
  FR_TRI_CASES(FR_CALL)
#undef FR_CALL
}

}  // namespace fr
