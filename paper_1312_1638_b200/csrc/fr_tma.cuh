// Shared pieces of the TMA-pipelined hexahedral kernels (fr_hex_tma.cu, fr_hex_fluxdiv_tma.cu): PTX wrappers for
// mbarriers and bulk tensor copies (sm_100a), the tensor-map encoder fetched through the runtime, launch helpers.
#pragma once
#include <cuda.h>  // CUtensorMap and its enums (types only: the encoder is fetched through the runtime)

#include <cstdint>
#include <cstdlib>

#include "fr_hex_tma.hpp"
#include "fr_ops1d.cuh"

namespace fr {
namespace {

constexpr int NV = 5;
constexpr size_t SMEM_MAX = 227 * 1024;

__host__ __device__ constexpr size_t al128(size_t x) { return (x + 127) / 128 * 128; }

// ---------------------------------------------------------------------------------------------
// PTX wrappers: mbarrier + bulk tensor copies
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_addr(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_addr(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_addr(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity) {
  const uint32_t a = smem_addr(bar);
  uint32_t ok;
  do {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n"
        : "=r"(ok)
        : "r"(a), "r"(parity)
        : "memory");
  } while (!ok);
}
// global load that the compiler may neither merge with an earlier load of the same address nor hoist
__device__ __forceinline__ double ld_nc_once(const double *p) {
  double v;
  asm volatile("ld.global.nc.f64 %0, [%1];" : "=d"(v) : "l"(p));
  return v;
}
__device__ __forceinline__ void fence_barrier_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void tma_load_3d(void *dst, const CUtensorMap *tm, int c0, int c1, int c2, uint64_t *bar) {
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];" ::"r"(
          smem_addr(dst)),
      "l"(tm), "r"(c0), "r"(c1), "r"(c2), "r"(smem_addr(bar))
      : "memory");
}

__device__ __forceinline__ void tma_load_4d(void *dst, const CUtensorMap *tm, int c0, int c1, int c2, int c3, uint64_t *bar) {
  asm volatile(
      "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];" ::"r"(
          smem_addr(dst)),
      "l"(tm), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(smem_addr(bar))
      : "memory");
}
__device__ __forceinline__ void tma_store_4d(const CUtensorMap *tm, int c0, int c1, int c2, int c3, const void *src) {
  asm volatile("cp.async.bulk.tensor.4d.global.shared::cta.bulk_group [%0, {%1, %2, %3, %4}], [%5];" ::"l"(tm), "r"(c0), "r"(c1),
               "r"(c2), "r"(c3), "r"(smem_addr(src))
               : "memory");
}
// bulk tensor store shared -> global (bulk async-group completion)
__device__ __forceinline__ void tma_store_3d(const CUtensorMap *tm, int c0, int c1, int c2, const void *src) {
  asm volatile("cp.async.bulk.tensor.3d.global.shared::cta.bulk_group [%0, {%1, %2, %3}], [%4];" ::"l"(tm), "r"(c0), "r"(c1), "r"(c2),
               "r"(smem_addr(src))
               : "memory");
}
__device__ __forceinline__ void tma_store_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void tma_store_wait_all() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }
__device__ __forceinline__ void tma_store_wait_read() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }

// per-thread asynchronous copies global -> shared (gathers): BYTES = 4 | 8 | 16
template <int BYTES>
__device__ __forceinline__ void cp_async(void *dst, const void *src) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], %2;" ::"r"(smem_addr(dst)), "l"(src), "n"(BYTES) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int PENDING>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(PENDING) : "memory"); }

// resident CTAs per SM the kernel is compiled for: limited by shared memory, by >= `regs` registers per thread
constexpr int min_blocks(size_t smem, int threads, int regs = 128) {
  int by_smem = (int)((SMEM_MAX + 1024) / (smem + 1024));
  int warps = (threads + 31) / 32;
  int by_regs = 65536 / (regs * 32 * warps);
  int by_thr = 2048 / (32 * warps);
  int m = by_smem < by_regs ? by_smem : by_regs;
  m = m < by_thr ? m : by_thr;
  return m < 1 ? 1 : (m > 8 ? 8 : m);
}

// Q~ -> Q at one solution point for variable a:  q_n = (1/J) sum_i S[i][n] q~_i   (Eq 10 :206)
template <typename R>
__device__ __forceinline__ void to_physical(const R (*S)[3], R rj, R qx, R qy, R qz, R *q) {
#pragma unroll
  for (int n = 0; n < 3; ++n) q[n] = rj * fma(S[0][n], qx, fma(S[1][n], qy, S[2][n] * qz));
}

// n . f_vis (Eq 22-24) from the perturbation state w and its gradient fed one variable at a time (getg(a, g) -> d_n w_a), so
// that at most the velocity-gradient tensor is live: d_i v_j by the quotient rule with dv = w_m / rho, Delta dT = (mu gamma / Pr)
// d e (A8); formulas of subtract_viscous_flux (fr_physics.cuh).
template <typename R, typename GetG>
__device__ __forceinline__ void visc_normal_stream(const R *w, const R *nrm, const Phys &ph, GetG getg, R *G) {
  const R rrho = (R)1 / (w[0] + (R)ph.rho0), Es = (w[4] - (R)ph.p0) * rrho;
  const R mu = (R)ph.mu;
  R v[3], dvl[3], g0[3], dv[3][3], de[3];
#pragma unroll
  for (int d = 0; d < 3; ++d) { dvl[d] = w[1 + d] * rrho; v[d] = (R)ph.v0[d] + dvl[d]; }
#pragma unroll
  for (int a = 0; a < NV; ++a) {
    R g[3];
    getg(a, g);
#pragma unroll
    for (int n = 0; n < 3; ++n) {
      if (a == 0) g0[n] = g[n];
      else if (a < 4) dv[n][a - 1] = (g[n] - dvl[a - 1] * g0[n]) * rrho;
      else de[n] = (g[n] - Es * g0[n]) * rrho;
    }
  }
  const R lam = (R)(-2.0 / 3.0) * mu * (dv[0][0] + dv[1][1] + dv[2][2]);
  const R kap = (R)(ph.mu * ph.gamma / ph.Pr);
  R Tm[3][3];
#pragma unroll
  for (int a = 0; a < 3; ++a)
#pragma unroll
    for (int b = 0; b < 3; ++b) Tm[a][b] = mu * (dv[a][b] + dv[b][a]) + (a == b ? lam : (R)0);
  G[0] = 0;
#pragma unroll
  for (int b = 0; b < 3; ++b) G[1 + b] = fma(nrm[0], Tm[0][b], fma(nrm[1], Tm[1][b], nrm[2] * Tm[2][b]));
  R s = 0;
#pragma unroll
  for (int n = 0; n < 3; ++n) {
    R d = de[n], vt = 0;
#pragma unroll
    for (int b = 0; b < 3; ++b) { d -= v[b] * dv[n][b]; vt += v[b] * Tm[b][n]; }
    s = fma(nrm[n], vt + kap * d, s);
  }
  G[4] = s;
}

// G at one flux point from the interpolated perturbation state and its gradient.  Interior: n . f_vis(w^f, q^f) with the
// element's own outward normal (the pair kernel applies the LDG weights 1/2 +- beta, Eq 27).  Boundary:
// the complete (1/2+beta) n.f_vis(u_L, q_L) + (1/2-beta) n.f_vis(B_ldg u_L, B_ldg q_L)  (App C, A20).
template <bool BND>
__device__ __forceinline__ void face_visc(const double *wf, const double (*qf)[NV], const double *nrm, const Phys &ph, int pe,
                                          const BcDev *__restrict__ bcs, double *G) {
  normal_viscous_flux<3>(wf, qf, nrm, ph, G);
  if (BND && pe < 0) {
    double uf[NV], gi[NV], gl[NV], qg[3][NV], GR[NV];
    from_pert<3>(ph, wf, uf);
    const double keep = ghost_states<3>(bcs[-1 - pe], uf, ph.gamma, gi, gl);
    to_pert<3>(ph, gl, gl);
#pragma unroll
    for (int n = 0; n < 3; ++n)
#pragma unroll
      for (int a = 0; a < NV; ++a) qg[n][a] = keep * qf[n][a];
    normal_viscous_flux<3>(gl, qg, nrm, ph, GR);
    const double wl = 0.5 + ph.beta, wr = 0.5 - ph.beta;
#pragma unroll
    for (int a = 0; a < NV; ++a) G[a] = (wl != 0.0 ? wl * G[a] : 0.0) + (wr != 0.0 ? wr * GR[a] : 0.0);
  }
}

// the same with operands in R (boundary instantiations of k_hex_gradface; the ghost-state algebra stays in double)
template <bool BND, typename R>
__device__ __forceinline__ void face_visc_r(const R *wf, const R (*qf)[NV], const R *nrm, const Phys &ph, int pe, const BcDev *__restrict__ bcs,
                                            R *G) {
  double w[NV], q[3][NV], n3[3], g[NV];
#pragma unroll
  for (int a = 0; a < NV; ++a) w[a] = (double)wf[a];
#pragma unroll
  for (int n = 0; n < 3; ++n) {
    n3[n] = (double)nrm[n];
#pragma unroll
    for (int a = 0; a < NV; ++a) q[n][a] = (double)qf[n][a];
  }
  face_visc<BND>(w, q, n3, ph, pe, bcs, g);
#pragma unroll
  for (int a = 0; a < NV; ++a) G[a] = (R)g[a];
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                  const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encoder() {
  static EncodeTiledFn fn = [] {
    void *p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) != cudaSuccess || q != cudaDriverEntryPointSuccess)
      p = nullptr;
    return (EncodeTiledFn)p;
  }();
  return fn;
}

// 3-D view (d0 = elements (contiguous), d1 = rows, d2 = blocks of rows); strides in elements
bool encode3(CUtensorMap *m, bool f64, const void *base, uint64_t d0, uint64_t d1, uint64_t d2, uint64_t s1, uint64_t s2, uint32_t b0,
             uint32_t b1, uint32_t b2) {
  EncodeTiledFn fn = encoder();
  if (!fn) return false;
  const uint64_t esz = f64 ? 8 : 4;
  cuuint64_t dims[3] = {d0, d1, d2};
  cuuint64_t strides[2] = {s1 * esz, s2 * esz};
  cuuint32_t box[3] = {b0, b1, b2};
  cuuint32_t estr[3] = {1, 1, 1};
  CUresult r = fn(m, f64 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, const_cast<void *>(base), dims, strides,
                  box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                  CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return r == CUDA_SUCCESS;
}

// Element-blocked internal array (fr_dev.hpp: fp_row) [ld / FR_BLK][r2][r1][FR_BLK] as a 4-D map (lane, r1, r2, block);
// box (E, b1, b2, 1).  Coordinates of a CTA that starts at element e0: (e0 % FR_BLK, row, block of rows, e0 / FR_BLK).
inline bool encode_blk(CUtensorMap *m, bool f64, const void *base, uint64_t ld, uint64_t r1, uint64_t r2, uint32_t E, uint32_t b1, uint32_t b2,
                       int bcast = 0) {
  EncodeTiledFn fn = encoder();
  if (!fn) return false;
  const uint64_t esz = f64 ? 8 : 4;
  cuuint64_t dims[4] = {(cuuint64_t)FR_BLK, r1, r2, ld / FR_BLK};
  cuuint64_t strides[3] = {(cuuint64_t)FR_BLK * esz, r1 * FR_BLK * esz, r1 * r2 * FR_BLK * esz};
  // affine meshes store one point per element: the point dimension(s) are broadcast through a zero stride, so the
  // kernels see the same [rows][E] boxes while DRAM holds (and serves) each value once
  if (bcast == 1) { strides[0] = 0; strides[1] = FR_BLK * esz; strides[2] = r2 * FR_BLK * esz; }   // r1 broadcast: [block][r2][FR_BLK]
  if (bcast == 2) { strides[0] = 0; strides[1] = 0; strides[2] = FR_BLK * esz; }                    // r1 and r2 broadcast: [block][FR_BLK]
  cuuint32_t box[4] = {E, b1, b2, 1};
  cuuint32_t estr[4] = {1, 1, 1, 1};
  return fn(m, f64 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, const_cast<void *>(base), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
            CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// function attributes are per device: one flag per (kernel instantiation, device ordinal)
// Encoded tensor maps of one context, keyed on (kernel, the pointers a call passes): cuTensorMapEncodeTiled costs about a
// microsecond per map and an RHS needs 11 of them, which matters for the launch-bound small cases; RK steppers alternate
// between two or three pointer sets.
struct MapCache {
  struct Ent { int id = -1; const void *p[3] = {nullptr, nullptr, nullptr}; CUtensorMap m[6]; };
  static const int CAP = 16;
  Ent e[CAP];
  int next = 0;
  // returns the entry and whether it has to be filled
  Ent *get(int id, const void *a, const void *b, const void *c, bool &fresh) {
    for (int i = 0; i < CAP; ++i)
      if (e[i].id == id && e[i].p[0] == a && e[i].p[1] == b && e[i].p[2] == c) { fresh = false; return &e[i]; }
    Ent *x = &e[next];
    next = (next + 1) % CAP;
    x->id = id; x->p[0] = a; x->p[1] = b; x->p[2] = c;
    fresh = true;
    return x;
  }
};

template <typename K>
cudaError_t set_smem(K kern, size_t smem, DevFlags &done, int dev) {
  if (done.test(dev)) return cudaSuccess;
  cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
  if (e == cudaSuccess) done.set(dev);
  return e;
}

// Thread slot -> point (i, j) of a slice, grouping the points in 2 x 2 patches: the four slots that share a warp with E = 8
// elements then touch two x-lines and two y-lines instead of (up to) four distinct lines in one direction, so a line read in
// either direction is one 128-byte shared-memory wavefront.  A bijection of 0 .. N*N-1 that maps slots < k*N onto points < k*N
// only loosely; the kernels use it for nothing but the choice of (i, j).
template <int N>
__device__ __forceinline__ int patch_ij(int slot) {
  constexpr int M = N / 2;  // full 2 x 2 patches per patch row; a patch row holds 2 N points
  if (slot >= 2 * N * M) return (N - 1) * N + (slot - 2 * N * M);  // last point row of an odd N
  const int br = slot / (2 * N), s2 = slot % (2 * N);
  if (s2 < 4 * M) return (2 * br + ((s2 >> 1) & 1)) * N + 2 * (s2 >> 2) + (s2 & 1);
  return (2 * br + (s2 - 4 * M)) * N + N - 1;  // last point column of an odd N
}

// elements per CTA for each n = p + 1 (row segments of E*8 bytes; N = 7: only 4 elements fit the shared memory).  The same in
// single precision: twice the elements (64-byte segments again) halves the resident CTAs of the register-bound kernels and
// was slower (C3 fp32: gradient kernel 0.41 -> 0.47 ms, divergence kernel 0.19 -> 0.22 ms)
template <int N, typename T>
struct Cfg {
  static constexpr int E = N <= 2 ? 32 : (N == 3 ? 16 : (N <= 6 ? 8 : 4));
  // the two z-slab kernels at p = 5 in double precision: 8 elements leave room for ONE resident CTA of 9 warps, 4 elements for
  // two of 5 (48^3 elements: gradient kernel 2.41 -> 2.34 ms, divergence kernel 1.41 -> 1.31 ms)
  static constexpr int E_SLAB = (N == 6 && sizeof(T) == 8) ? 4 : E;
};

}  // namespace
}  // namespace fr
