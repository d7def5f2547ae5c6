// Tensor-product (sum-factorised) kernels for quadrilateral / hexahedral elements.
//
// On tensor-product elements every row of M0, M4, M1, M3, M6 touches one line of
// n = p+1 solution points (plus the two flux points at its ends), so the dense App-A GEMMs of the paper
// (2*N_V*(8 N_f N_u + 6 N_u^2) flop per element) collapse to N_V*(12 n^4 + 72 n^3): the path becomes
// HBM-bound.  The paper anticipates "bespoke matrix multiply kernels" (:282).
//
// Layout: every state matrix is [row][variable][ld], element fastest; a warp covers 32
// consecutive columns (variable, element) of one row, so every global access is a fully used 256-byte row
// segment.  Threads own output points and gather the n values of each line through L1 (a CTA covers all
// rows of its 32 columns, so each input is fetched from L2/HBM once per CTA).
// The 1-D operators travel as a kernel parameter (constant bank, uniform broadcast reads).
#include "fr_tensor.hpp"
#include "fr_hex_tma.hpp"
#include "fr_ops1d.cuh"

#include <cstdlib>

namespace fr {
namespace {


// rho of point m on the line through (direction d, face-point index idx)
template <int N, int ND>
__device__ __forceinline__ int line_base(int d, int idx, int &stride) {
  if (ND == 2) {
    stride = d == 0 ? 1 : N;
    return d == 0 ? N * idx : idx;
  }
  const int a = idx % N, b = idx / N;
  if (d == 0) { stride = 1; return N * a + N * N * b; }
  if (d == 1) { stride = N; return a + N * N * b; }
  stride = N * N;
  return a + N * b;
}

// U^f = M0 U (Eq 6 / Eq 41) and, with nblk = ND, Q^f = M5 Q (Eq 11 / Eq 43).
template <int N, int ND, typename TIN>
__global__ void __launch_bounds__(1024) k_tp_interp(Ops1D<N> op, const TIN *__restrict__ in, double *__restrict__ out, int64_t ncols,
                                                    int64_t ld, int64_t Nel, int64_t in_blk, int64_t out_blk) {
  constexpr int NFP = ipow(N, ND - 1);
  const int64_t col = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (col >= ncols || (col % ld) >= Nel) return;
  in += (size_t)blockIdx.z * in_blk + col;
  const size_t rs = (size_t)ncols;  // distance between consecutive flux points: out[fp][a][ld]
  out += (size_t)blockIdx.z * out_blk + col;
  for (int idx = threadIdx.y; idx < NFP; idx += blockDim.y) {
#pragma unroll
    for (int d = 0; d < ND; ++d) {
      int stride;
      const int base = line_base<N, ND>(d, idx, stride);
      double sm = 0, sp = 0;
#pragma unroll
      for (int m = 0; m < N; ++m) {
        const double v = (double)in[(size_t)(base + m * stride) * ncols];
        sm = fma(op.lm[m], v, sm);
        sp = fma(op.lp[m], v, sp);
      }
      out[(size_t)((2 * d) * NFP + idx) * rs] = sm;
      out[(size_t)((2 * d + 1) * NFP + idx) * rs] = sp;
    }
  }
}

// Q = J^-T {M4 U + M6 (C - U^f)}  (Eq 9-10 / Eq 42): thread per solution point and element, looping over
// the variables so that S and 1/J are loaded once.  jump = C - U^f at the flux points.
template <int N, int ND, typename TIN>
__global__ void __launch_bounds__(256) k_tp_grad(Ops1D<N> op, const TIN *__restrict__ u, const double *__restrict__ jump,
                                                  const double *__restrict__ smat, const double *__restrict__ rcpj,
                                                  double *__restrict__ q, int64_t ncols, int64_t ld, int64_t Nel) {
  constexpr int NU = ipow(N, ND), NFP = ipow(N, ND - 1), NV = ND + 2;
  const int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= Nel) return;
  u += e; jump += e; q += e;
  for (int r = threadIdx.y; r < NU; r += blockDim.y) {
    int ii[3];
    ii[0] = r % N; ii[1] = (r / N) % N; ii[2] = ND == 3 ? r / (N * N) : 0;
    double S[ND][ND];
#pragma unroll
    for (int i = 0; i < ND; ++i)
#pragma unroll
      for (int n = 0; n < ND; ++n) S[i][n] = smat[((size_t)(i * ND + n) * NU + r) * ld + e];
    const double rj = rcpj[(size_t)r * ld + e];
#pragma unroll 1
    for (int a = 0; a < NV; ++a) {
      double qt[ND];
#pragma unroll
      for (int d = 0; d < ND; ++d) {
        const int stride = d == 0 ? 1 : (d == 1 ? N : N * N);
        const int base = r - ii[d] * stride;
        // face-point index of this line: the remaining tensor indices, lowest fastest
        int idx;
        if (ND == 2) idx = d == 0 ? ii[1] : ii[0];
        else idx = d == 0 ? ii[1] + N * ii[2] : (d == 1 ? ii[0] + N * ii[2] : ii[0] + N * ii[1]);
        double s = 0;
#pragma unroll
        for (int m = 0; m < N; ++m) s = fma(op.D[ii[d] * N + m], (double)u[(size_t)(base + m * stride) * ncols + a * ld], s);
        // M6 = n~ (x) M3 (A1): the reference normal is -1 on the -1 face
        s = fma(-op.gm[ii[d]], jump[(size_t)((2 * d) * NFP + idx) * ncols + a * ld], s);
        s = fma(op.gp[ii[d]], jump[(size_t)((2 * d + 1) * NFP + idx) * ncols + a * ld], s);
        qt[d] = s;
      }
#pragma unroll
      for (int n = 0; n < ND; ++n) {
        double s = 0;
#pragma unroll
        for (int i = 0; i < ND; ++i) s = fma(S[i][n], qt[i], s);
        q[(size_t)(n * NU + r) * ncols + a * ld] = s * rj;
      }
    }
  }
}

// R = -(1/J) {(M1 - M3 M2) F~ + M3 D~}  (Eq 18-19 / Eq 44): thread per solution point and column.
template <int N, int ND, typename TOUT>
__global__ void __launch_bounds__(1024) k_tp_div(Ops1D<N> op, const double *__restrict__ ft, const double *__restrict__ dt,
                                                 const double *__restrict__ rcpj, TOUT *__restrict__ rhs, int64_t ncols, int64_t ld,
                                                 int64_t Nel) {
  constexpr int NU = ipow(N, ND), NFP = ipow(N, ND - 1);
  const int64_t col = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (col >= ncols) return;
  const int64_t e = col % ld;
  if (e >= Nel) return;
  ft += col; dt += col; rhs += col;
  for (int r = threadIdx.y; r < NU; r += blockDim.y) {
    int ii[3];
    ii[0] = r % N; ii[1] = (r / N) % N; ii[2] = ND == 3 ? r / (N * N) : 0;
    double acc = 0;
#pragma unroll
    for (int d = 0; d < ND; ++d) {
      const int stride = d == 0 ? 1 : (d == 1 ? N : N * N);
      const int base = r - ii[d] * stride;
      int idx;
      if (ND == 2) idx = d == 0 ? ii[1] : ii[0];
      else idx = d == 0 ? ii[1] + N * ii[2] : (d == 1 ? ii[0] + N * ii[2] : ii[0] + N * ii[1]);
      const double *f = ft + (size_t)d * NU * ncols;
#pragma unroll
      for (int m = 0; m < N; ++m) acc = fma(op.Dh[ii[d] * N + m], f[(size_t)(base + m * stride) * ncols], acc);
      acc = fma(op.gm[ii[d]], dt[(size_t)((2 * d) * NFP + idx) * ncols], acc);
      acc = fma(op.gp[ii[d]], dt[(size_t)((2 * d + 1) * NFP + idx) * ncols], acc);
    }
    rhs[(size_t)r * ncols] = (TOUT)(-acc * rcpj[(size_t)r * ld + e]);
  }
}

template <int N, int ND, typename T>
cudaError_t run(const DevConsts &c, const TensorPlan &tp, const T *u, T *rhs, char *work, cudaStream_t s, Prof *prof) {
  constexpr int NU = ipow(N, ND), NFP = ipow(N, ND - 1), NF = 2 * ND * NFP;
  double *uf = (double *)(work + tp.off_uf), *cf = (double *)(work + tp.off_cf), *qu = (double *)(work + tp.off_qu),
         *qf = (double *)(work + tp.off_qf);
  if constexpr (ND == 3) {
    // hexahedra: sm_100a TMA path, 4 launches for Navier-Stokes (3 for Euler); C^f, Q^f and F~ are never stored; the
    // flux-point arrays and Q are in the storage precision T
    (void)cf;
    FR_MARK(prof, "hex_interp_tma");
    cudaError_t e = hex_tma_interp(c, tp.h_ops, u, uf, s);
    if (e != cudaSuccess) return e;
    if (c.ns) {
      FR_MARK(prof, "hex_gradface");
      e = hex_tma_gradface(c, tp.h_ops, u, uf, qu, qf, s);
      if (e != cudaSuccess) return e;
      FR_MARK(prof, "common_flux_g");
      launch_common_flux_g(c, uf, qu, !c.f64, s);
    } else {
      FR_MARK(prof, "common_flux");
      launch_common_flux(c, uf, qf, !c.f64, s);
    }
    FR_MARK(prof, "hex_fluxdiv_tma");
    e = hex_tma_fluxdiv(c, tp.h_ops, u, qf, uf, rhs, s);
    return e != cudaSuccess ? e : cudaGetLastError();
  } else {
    // quadrilaterals (p = 0 and p >= 5; lower orders run the fused element kernels): L1-gather line kernels
    const Ops1D<N> op = make_ops<N>(tp.h_ops);
    const int64_t ncols = (int64_t)c.NV * c.ld;
    constexpr int LW = 32;  // lanes (columns) per CTA row
    const int rows = 1024 / LW;
    const unsigned gx = (unsigned)((ncols + LW - 1) / LW), ge = (unsigned)((c.Nel + LW - 1) / LW);
    const dim3 bf(LW, NFP < rows ? NFP : rows), bu(LW, NU < rows ? NU : rows);
    FR_MARK(prof, "tp_interp");
    k_tp_interp<N, ND, T><<<dim3(gx, 1, 1), bf, 0, s>>>(op, u, uf, ncols, c.ld, c.Nel, 0, 0);
    if (c.ns) {
      FR_MARK(prof, "common_sol");
      launch_common_jump(c, uf, cf, s);
      FR_MARK(prof, "tp_grad");
      k_tp_grad<N, ND, T><<<dim3(ge, 1, 1), dim3(LW, 256 / LW), 0, s>>>(op, u, cf, c.smat, c.rcpj, qu, ncols, c.ld, c.Nel);
      FR_MARK(prof, "tp_interp_q");
      k_tp_interp<N, ND, double><<<dim3(gx, 1, ND), bf, 0, s>>>(op, qu, qf, ncols, c.ld, c.Nel, (int64_t)NU * ncols, (int64_t)NF * ncols);
    }
    FR_MARK(prof, "tflux");
    launch_tflux(c, u, qu, s);
    FR_MARK(prof, "common_flux");
    launch_common_flux(c, uf, qf, false, s);
    FR_MARK(prof, "tp_div");
    k_tp_div<N, ND, T><<<dim3(gx, 1, 1), bu, 0, s>>>(op, qu, uf, c.rcpj, rhs, ncols, c.ld, c.Nel);
    return cudaGetLastError();
  }
}

template <int ND>
cudaError_t dispatch_n(const DevConsts &c, const TensorPlan &tp, const void *u, void *rhs, char *work, cudaStream_t s, Prof *prof) {
#define FR_CASE(NN)                                                                                              \
  case NN:                                                                                                       \
    return c.f64 ? run<NN, ND, double>(c, tp, (const double *)u, (double *)rhs, work, s, prof)                    \
                 : run<NN, ND, float>(c, tp, (const float *)u, (float *)rhs, work, s, prof);
  switch (c.n) {
    FR_CASE(1) FR_CASE(2) FR_CASE(3) FR_CASE(4) FR_CASE(5) FR_CASE(6) FR_CASE(7) FR_CASE(8)
    default: return cudaErrorNotSupported;
  }
#undef FR_CASE
}

}  // namespace

// quadrilaterals at any order 0 <= p <= 7; hexahedra when the TMA kernels can run (c.blk: decided in fr_api.cu with the layout)
bool tensor_supported(const DevConsts &c) {
  if (c.n < 1 || c.n > 8) return false;
  return c.etype == FR_QUAD || (c.etype == FR_HEX && c.blk);
}

cudaError_t tensor_plan(const DevConsts &c, const RefOps &o, const MeshConsts &, TensorPlan &tp, std::vector<void *> &) {
  tp = TensorPlan();
  const int n = o.n;
  double *p = tp.h_ops;
  for (int i = 0; i < n * n; ++i) *p++ = o.D1[i];
  for (int i = 0; i < n * n; ++i) *p++ = o.Dhat[i];
  for (int i = 0; i < n; ++i) *p++ = o.lm[i];
  for (int i = 0; i < n; ++i) *p++ = o.lp[i];
  for (int i = 0; i < n; ++i) *p++ = o.gm[i];
  for (int i = 0; i < n; ++i) *p++ = o.gp[i];
  auto al = [](int64_t x) { return (x + 255) / 256 * 256; };
  const int64_t ncols = (int64_t)c.NV * c.ld;
  int64_t off = 0;
  tp.use_tma = c.blk;
  if (tp.use_tma) {  // U^f -> D~, G^f and Q (slice-major) in the storage precision
    const int64_t esz = c.f64 ? 8 : 4;
    tp.off_uf = off; off = al(off + (int64_t)o.Nf * ncols * esz);
    tp.off_cf = off;
    tp.off_qu = off; if (c.ns) off = al(off + (int64_t)o.Nf * ncols * esz);
    tp.off_qf = off; if (c.ns) off = al(off + (int64_t)o.nd * o.Nu * ncols * esz);
  } else {
    tp.off_uf = off; off = al(off + (int64_t)o.Nf * ncols * 8);
    tp.off_cf = off; if (c.ns) off = al(off + (int64_t)o.Nf * ncols * 8);
    tp.off_qu = off; off = al(off + (int64_t)o.nd * o.Nu * ncols * 8);
    tp.off_qf = off; if (c.ns) off = al(off + (int64_t)o.nd * o.Nf * ncols * 8);
  }
  tp.work_bytes = off;
  return cudaSuccess;
}

cudaError_t tensor_rhs(const DevConsts &c, const TensorPlan &tp, const void *u, void *rhs, char *work, cudaStream_t s, Prof *prof) {
  return c.nd == 2 ? dispatch_n<2>(c, tp, u, rhs, work, s, prof) : dispatch_n<3>(c, tp, u, rhs, work, s, prof);
}

int tensor_rhs_launches(const DevConsts &c) {
  int n;
  if (c.nd == 3) n = c.ns ? 4 : 3;  // interp, (gradface,) common flux, fluxdiv
  else n = c.ns ? 7 : 4;            // interp, (common sol, grad, interp q,) tflux, common flux, div
  const int pair_groups = (c.nd == 3 || !c.ns) ? 1 : 2;  // launch groups that run over flux-point pairs / boundary points
  if (c.nbnd) n += pair_groups;
  if (!c.npairs) n -= pair_groups;
  return n;
}

}  // namespace fr
