// TMA-fed, mbarrier-pipelined "z-slab" kernels for hexahedral elements (sm_100a).
//
// Two kernels carry parts (2b)-(7) of the Navier-Stokes right-hand side (BASELINE.json north_star):
//
//   k_hex_gradface : Q = J^-T {M4 U + M6 (C - U^f)} at the solution points (Eq 9-10 / Eq 42 :753), interpolated
//                    to the element's own flux points (Eq 11 / Eq 43 :764) and contracted at once with the
//                    outward unit normal: G^f = n . f_vis(U^f, Q^f)  (Eq 22-24, the viscous part of Eq 26-27).
//                    Only G^f (N_V values per flux point) goes to HBM: neither Q (3 N_V N_u) nor Q^f
//                    (3 N_V N_f) is ever stored.  Boundary flux points get the complete LDG viscous flux
//                    with the ghost state of App C.
//   k_hex_rhs_tma  : recomputes Q from U and the interface jumps, F~ = S f(U, Q) (Eq 12), then
//                    R = -(1/J) {(M1 - M3 M2) F~ + M3 D~}  (Eq 18-19 / Eq 44 :772).  Euler: no gradient part.
//
// Data movement: a CTA owns E consecutive elements.  The U block of those elements ([N_u*N_V] rows of E
// values) is brought into shared memory by ONE 3-D TMA box load; the metric terms S (9 rows per point), 1/J
// and the x/y-face jumps stream slice by slice (z = k) through a two-stage ring of TMA box loads completing on
// mbarriers, issued two slices ahead by one thread, so HBM latency is covered without registers or occupancy.
// Thread (e, i, j) owns the column of points (i, j, .); contractions along x and y read shared memory,
// contractions along z use operator entries from the constant bank.
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
__device__ __forceinline__ void fence_barrier_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void tma_load_3d(void *dst, const CUtensorMap *tm, int c0, int c1, int c2, uint64_t *bar) {
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];" ::"r"(
          smem_addr(dst)),
      "l"(tm), "r"(c0), "r"(c1), "r"(c2), "r"(smem_addr(bar))
      : "memory");
}

// ---------------------------------------------------------------------------------------------
// shared-memory layouts (byte offsets from a 128-byte aligned base)
// ---------------------------------------------------------------------------------------------
template <int N, int E, bool NS, typename T, int NB>
struct RhsLay {
  static constexpr int NFP = N * N, NU = N * NFP;
  static constexpr size_t BAR = 0;
  static constexpr size_t OPS = 128;  // sD, sDh
  static constexpr size_t U = OPS + al128(2 * N * N * 8);
  static constexpr uint32_t U_TX = NU * NV * E * sizeof(T);
  static constexpr size_t RJ = U + al128(U_TX);
  static constexpr uint32_t RJ_TX = NU * E * 8;
  static constexpr size_t ST = RJ + al128(RJ_TX);
  static constexpr uint32_t S_TX = 9 * NFP * E * 8, J_TX = NS ? 4 * N * NV * E * 8 : 0;
  static constexpr size_t ST_J = al128(S_TX);
  static constexpr size_t ST_BYTES = ST_J + al128(J_TX);
  static constexpr size_t F = ST + 2 * ST_BYTES;
  static constexpr size_t F_BYTES = 2 * NV * NFP * E * 8;
  static constexpr size_t TOTAL = F + NB * F_BYTES + 128;  // + slack for the manual 128-byte alignment
};

template <int N, int E, typename T>
struct GfLay {
  static constexpr int NFP = N * N, NU = N * NFP;
  static constexpr size_t BAR = 0;
  static constexpr size_t OPS = 128;  // sD [N*N], sL [2][N]
  static constexpr size_t U = OPS + al128((N * N + 2 * N) * 8);
  static constexpr uint32_t U_TX = NU * NV * E * sizeof(T);
  static constexpr size_t ST = U + al128(U_TX);
  static constexpr uint32_t S_TX = 9 * NFP * E * 8, R_TX = NFP * E * 8, J_TX = 4 * N * NV * E * 8;
  static constexpr size_t ST_R = al128(S_TX);
  static constexpr size_t ST_J = ST_R + al128(R_TX);
  static constexpr size_t ST_BYTES = ST_J + al128(J_TX);
  static constexpr size_t Q = ST + 2 * ST_BYTES;
  static constexpr size_t Q_BYTES = 3 * NV * NFP * E * 8;
  static constexpr size_t TOTAL = Q + Q_BYTES + 128;
};

// resident CTAs per SM the kernel is compiled for: limited by shared memory, by >= 128 registers per thread
constexpr int min_blocks(size_t smem, int threads) {
  int by_smem = (int)((SMEM_MAX + 1024) / (smem + 1024));
  int warps = (threads + 31) / 32;
  int by_regs = 65536 / (128 * 32 * warps);
  int by_thr = 2048 / (32 * warps);
  int m = by_smem < by_regs ? by_smem : by_regs;
  m = m < by_thr ? m : by_thr;
  return m < 1 ? 1 : (m > 8 ? 8 : m);
}

// Q~ -> Q at one solution point for variable a:  q_n = (1/J) sum_i S[i][n] q~_i   (Eq 10 :206)
__device__ __forceinline__ void to_physical(const double (*S)[3], double rj, double qx, double qy, double qz, double *q) {
#pragma unroll
  for (int n = 0; n < 3; ++n) q[n] = rj * fma(S[0][n], qx, fma(S[1][n], qy, S[2][n] * qz));
}

// F~ = S f(u, q) at one point (Eq 12 :214 with Eq 20-24)
template <bool NS>
__device__ __forceinline__ void point_tflux(const double *uu, const double (*qq)[NV], const double (*S)[3], const Phys &ph,
                                            double (*F)[NV]) {
  double f[3][NV], v[3], p;
  inviscid_flux<3>(uu, ph.gamma, f, v, p);
  if (NS) subtract_viscous_flux<3>(uu, qq, v, ph, f);
#pragma unroll
  for (int i = 0; i < 3; ++i)
#pragma unroll
    for (int a = 0; a < NV; ++a) F[i][a] = fma(S[i][0], f[0][a], fma(S[i][1], f[1][a], S[i][2] * f[2][a]));
}

// ---------------------------------------------------------------------------------------------
// k_hex_rhs_tma
// ---------------------------------------------------------------------------------------------
// tmU: u as (ld, NFP*NV, N), box (E, NFP*NV, N);  tmS: smat as (ld, NU, 9), box (E, NFP, 9);
// tmR: rcpj as (ld, NFP, N), box (E, NFP, N);      tmJ: jump as (ld, NFP*NV, 6), box (E, N*NV, 4).
template <int N, int E, bool NS, typename T, int NB, int MINB>
__global__ void __launch_bounds__(N *N *E, MINB)
    k_hex_rhs_tma(const __grid_constant__ CUtensorMap tmU, const __grid_constant__ CUtensorMap tmS,
                  const __grid_constant__ CUtensorMap tmR, const __grid_constant__ CUtensorMap tmJ, Ops1D<N> op, Phys ph,
                  const double *__restrict__ jump, const double *__restrict__ dt, T *__restrict__ rhs, int64_t ld, int64_t Nel) {
  using L = RhsLay<N, E, NS, T, NB>;
  constexpr int NFP = N * N;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  unsigned char *sm = smem_raw + ((128u - (smem_addr(smem_raw) & 127u)) & 127u);  // stays in the shared address space
  uint64_t *bar = (uint64_t *)(sm + L::BAR);  // [0]: U block + 1/J block, [1], [2]: stages
  double *sD = (double *)(sm + L::OPS), *sDh = sD + N * N;
  const T *sU = (const T *)(sm + L::U);            // [NU*NV][E], row = (NFP k + ij) NV + a
  const double *sRJ = (const double *)(sm + L::RJ);  // [NU][E]
  unsigned char *sSt = sm + L::ST;
  double *sF = (double *)(sm + L::F);              // [NB][2][NV][NFP][E]
  const int tid = threadIdx.x, el = tid % E, ij = tid / E, i = ij % N, j = ij / N;
  const int e0 = blockIdx.x * E;
  const int64_t e = (int64_t)e0 + el;
  const bool act = e < Nel;

  if (tid == 0) {
    mbar_init(&bar[0], 1); mbar_init(&bar[1], 1); mbar_init(&bar[2], 1);
    fence_barrier_init();
    fence_proxy_async();
  }
  for (int t = tid; t < N * N; t += NFP * E) { sD[t] = op.D[t]; sDh[t] = op.Dh[t]; }
  __syncthreads();
  auto issue_stage = [&](int s, int k) {
    mbar_expect_tx(&bar[1 + s], L::S_TX + L::J_TX);
    tma_load_3d(sSt + s * L::ST_BYTES, &tmS, e0, NFP * k, 0, &bar[1 + s]);
    if (NS) tma_load_3d(sSt + s * L::ST_BYTES + L::ST_J, &tmJ, e0, N * k * NV, 0, &bar[1 + s]);
  };
  if (tid == 0) {
    mbar_expect_tx(&bar[0], L::U_TX + L::RJ_TX);
    tma_load_3d(sm + L::U, &tmU, e0, 0, 0, &bar[0]);
    tma_load_3d(sm + L::RJ, &tmR, e0, 0, 0, &bar[0]);
    issue_stage(0, 0);
    if (N > 1) issue_stage(1, 1);
  }
  double jzm[NV], jzp[NV];
  if (NS) {
#pragma unroll
    for (int a = 0; a < NV; ++a) {
      jzm[a] = jump[((size_t)(4 * NFP + ij) * NV + a) * ld + e];
      jzp[a] = jump[((size_t)(5 * NFP + ij) * NV + a) * ld + e];
    }
  }
  const double gmi = op.gm[i], gpi = op.gp[i], gmj = op.gm[j], gpj = op.gp[j];
  double acc[N][NV];
#pragma unroll
  for (int k = 0; k < N; ++k)
#pragma unroll
    for (int a = 0; a < NV; ++a) acc[k][a] = 0.0;
  mbar_wait(&bar[0], 0);

#pragma unroll
  for (int k = 0; k < N; ++k) {
    mbar_wait(&bar[1 + (k & 1)], (k >> 1) & 1);
    const double *stS = (const double *)(sSt + (k & 1) * L::ST_BYTES);
    const double *stJ = (const double *)(sSt + (k & 1) * L::ST_BYTES + L::ST_J);
    double F[3][NV];
    {
      double S[3][3], uu[NV], qq[3][NV];
#pragma unroll
      for (int a = 0; a < 3; ++a)
#pragma unroll
        for (int b = 0; b < 3; ++b) S[a][b] = stS[((a * 3 + b) * NFP + ij) * E + el];
      const T *su = sU + (size_t)(NFP * k) * NV * E + el;  // slice k
#pragma unroll
      for (int a = 0; a < NV; ++a) uu[a] = (double)su[(ij * NV + a) * E];
      if (NS) {
        const double rj = sRJ[(NFP * k + ij) * E + el];
#pragma unroll
        for (int a = 0; a < NV; ++a) {
          // M6 = n~ (x) M3 (A1): the reference normal is -1 on the -1 faces
          double qx = fma(gpi, stJ[((1 * N + j) * NV + a) * E + el], -gmi * stJ[((0 * N + j) * NV + a) * E + el]);
          double qy = fma(gpj, stJ[((3 * N + i) * NV + a) * E + el], -gmj * stJ[((2 * N + i) * NV + a) * E + el]);
          double qz = fma(op.gp[k], jzp[a], -op.gm[k] * jzm[a]);
#pragma unroll
          for (int m = 0; m < N; ++m) {
            qx = fma(sD[i * N + m], (double)su[((j * N + m) * NV + a) * E], qx);
            qy = fma(sD[j * N + m], (double)su[((m * N + i) * NV + a) * E], qy);
            qz = fma(op.D[k * N + m], (double)sU[((size_t)(NFP * m + ij) * NV + a) * E + el], qz);
          }
          double q3[3];
          to_physical(S, rj, qx, qy, qz, q3);
          qq[0][a] = q3[0]; qq[1][a] = q3[1]; qq[2][a] = q3[2];
        }
      }
      point_tflux<NS>(uu, qq, S, ph, F);
    }
    double *buf = sF + (NB == 2 ? (k & 1) : 0) * (2 * NV * NFP * E);
    if (NB == 1 && k > 0) __syncthreads();  // the previous slice's contraction has finished reading sF
#pragma unroll
    for (int a = 0; a < NV; ++a) {
      buf[((0 * NV + a) * NFP + ij) * E + el] = F[0][a];
      buf[((1 * NV + a) * NFP + ij) * E + el] = F[1][a];
    }
    // z contraction: this point contributes to every point of its column
#pragma unroll
    for (int kk = 0; kk < N; ++kk)
#pragma unroll
      for (int a = 0; a < NV; ++a) acc[kk][a] = fma(op.Dh[kk * N + k], F[2][a], acc[kk][a]);
    __syncthreads();
    // every thread has consumed stage k&1: refill it with slice k+2
    if (tid == 0 && k + 2 < N) issue_stage(k & 1, k + 2);
    // x and y contractions within the slice
#pragma unroll
    for (int m = 0; m < N; ++m) {
      const double dx = sDh[i * N + m], dy = sDh[j * N + m];
#pragma unroll
      for (int a = 0; a < NV; ++a) {
        acc[k][a] = fma(dx, buf[((0 * NV + a) * NFP + j * N + m) * E + el], acc[k][a]);
        acc[k][a] = fma(dy, buf[((1 * NV + a) * NFP + m * N + i) * E + el], acc[k][a]);
      }
    }
  }
  if (!act) return;
  // lifting M3 D~ and the -1/J scale (Eq 19); faces: 0,1 = x-,x+ (idx j + N k); 2,3 = y (i + N k); 4,5 = z (i + N j)
  double dzm[NV], dzp[NV];
#pragma unroll
  for (int a = 0; a < NV; ++a) {
    dzm[a] = dt[((size_t)(4 * NFP + ij) * NV + a) * ld + e];
    dzp[a] = dt[((size_t)(5 * NFP + ij) * NV + a) * ld + e];
  }
#pragma unroll
  for (int k = 0; k < N; ++k) {
    const int r = ij + NFP * k;
    const double rj = sRJ[r * E + el];
    const int fx = j + N * k, fy = i + N * k;
#pragma unroll
    for (int a = 0; a < NV; ++a) {
      double v = acc[k][a];
      v = fma(op.gm[k], dzm[a], v);
      v = fma(op.gp[k], dzp[a], v);
      v = fma(gmi, dt[((size_t)(0 * NFP + fx) * NV + a) * ld + e], v);
      v = fma(gpi, dt[((size_t)(1 * NFP + fx) * NV + a) * ld + e], v);
      v = fma(gmj, dt[((size_t)(2 * NFP + fy) * NV + a) * ld + e], v);
      v = fma(gpj, dt[((size_t)(3 * NFP + fy) * NV + a) * ld + e], v);
      rhs[((size_t)r * NV + a) * ld + e] = (T)(-v * rj);
    }
  }
}

// ---------------------------------------------------------------------------------------------
// k_hex_gradface
// ---------------------------------------------------------------------------------------------
// G at one flux point from the interpolated state and gradient.  Interior: n . f_vis(u^f, q^f) with the
// element's own outward normal (the pair kernel applies the LDG weights 1/2 +- beta, Eq 27).  Boundary:
// the complete (1/2+beta) n.f_vis(u_L, q_L) + (1/2-beta) n.f_vis(B_ldg u_L, B_ldg q_L)  (App C, A20).
template <bool BND>
__device__ __forceinline__ void face_visc(const double *uf, const double (*qf)[NV], const double *nrm, const Phys &ph, int pe,
                                          const BcDev *__restrict__ bcs, double *G) {
  normal_viscous_flux<3>(uf, qf, nrm, ph, G);
  if (BND && pe < 0) {
    double gi[NV], gl[NV], qg[3][NV], GR[NV];
    const double keep = ghost_states<3>(bcs[-1 - pe], uf, ph.gamma, gi, gl);
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

// tmU, tmS, tmJ as above; tmR: rcpj as (ld, NFP, N), box (E, NFP, 1).
template <int N, int E, bool BND, typename T, int MINB>
__global__ void __launch_bounds__(N *N *E, MINB)
    k_hex_gradface(const __grid_constant__ CUtensorMap tmU, const __grid_constant__ CUtensorMap tmS,
                   const __grid_constant__ CUtensorMap tmR, const __grid_constant__ CUtensorMap tmJ, Ops1D<N> op, Phys ph,
                   const double *__restrict__ jump, const double *__restrict__ fp_n, const int32_t *__restrict__ fp_pe,
                   const BcDev *__restrict__ bcs, double *__restrict__ gf, int64_t ld, int64_t Nel) {
  using L = GfLay<N, E, T>;
  constexpr int NFP = N * N, NF = 6 * NFP;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  unsigned char *sm = smem_raw + ((128u - (smem_addr(smem_raw) & 127u)) & 127u);  // stays in the shared address space
  uint64_t *bar = (uint64_t *)(sm + L::BAR);
  double *sD = (double *)(sm + L::OPS), *sL = sD + N * N;  // sL[0][m] = l_m(-1), sL[1][m] = l_m(+1)
  const T *sU = (const T *)(sm + L::U);
  unsigned char *sSt = sm + L::ST;
  double *sQ = (double *)(sm + L::Q);  // [3*NV][NFP][E]
  const int tid = threadIdx.x, el = tid % E, ij = tid / E, i = ij % N, j = ij / N;
  const int e0 = blockIdx.x * E;
  const int64_t e = (int64_t)e0 + el;
  const bool act = e < Nel;

  if (tid == 0) {
    mbar_init(&bar[0], 1); mbar_init(&bar[1], 1); mbar_init(&bar[2], 1);
    fence_barrier_init();
    fence_proxy_async();
  }
  for (int t = tid; t < N * N; t += NFP * E) sD[t] = op.D[t];
  for (int t = tid; t < N; t += NFP * E) { sL[t] = op.lm[t]; sL[N + t] = op.lp[t]; }
  __syncthreads();
  auto issue_stage = [&](int s, int k) {
    mbar_expect_tx(&bar[1 + s], L::S_TX + L::R_TX + L::J_TX);
    tma_load_3d(sSt + s * L::ST_BYTES, &tmS, e0, NFP * k, 0, &bar[1 + s]);
    tma_load_3d(sSt + s * L::ST_BYTES + L::ST_R, &tmR, e0, 0, k, &bar[1 + s]);
    tma_load_3d(sSt + s * L::ST_BYTES + L::ST_J, &tmJ, e0, N * k * NV, 0, &bar[1 + s]);
  };
  if (tid == 0) {
    mbar_expect_tx(&bar[0], L::U_TX);
    tma_load_3d(sm + L::U, &tmU, e0, 0, 0, &bar[0]);
    issue_stage(0, 0);
    if (N > 1) issue_stage(1, 1);
  }
  double jzm[NV], jzp[NV];
#pragma unroll
  for (int a = 0; a < NV; ++a) {
    jzm[a] = jump[((size_t)(4 * NFP + ij) * NV + a) * ld + e];
    jzp[a] = jump[((size_t)(5 * NFP + ij) * NV + a) * ld + e];
  }
  const double gmi = op.gm[i], gpi = op.gp[i], gmj = op.gm[j], gpj = op.gp[j];
  double zm[3][NV], zp[3][NV];  // Q interpolated to the two z faces of this column
#pragma unroll
  for (int n = 0; n < 3; ++n)
#pragma unroll
    for (int a = 0; a < NV; ++a) zm[n][a] = zp[n][a] = 0.0;
  mbar_wait(&bar[0], 0);

#pragma unroll
  for (int k = 0; k < N; ++k) {
    mbar_wait(&bar[1 + (k & 1)], (k >> 1) & 1);
    const double *stS = (const double *)(sSt + (k & 1) * L::ST_BYTES);
    const double *stR = (const double *)(sSt + (k & 1) * L::ST_BYTES + L::ST_R);
    const double *stJ = (const double *)(sSt + (k & 1) * L::ST_BYTES + L::ST_J);
    const T *su = sU + (size_t)(NFP * k) * NV * E + el;  // slice k
    {
      double S[3][3];
#pragma unroll
      for (int a = 0; a < 3; ++a)
#pragma unroll
        for (int b = 0; b < 3; ++b) S[a][b] = stS[((a * 3 + b) * NFP + ij) * E + el];
      const double rj = stR[ij * E + el];
#pragma unroll
      for (int a = 0; a < NV; ++a) {
        double qx = fma(gpi, stJ[((1 * N + j) * NV + a) * E + el], -gmi * stJ[((0 * N + j) * NV + a) * E + el]);
        double qy = fma(gpj, stJ[((3 * N + i) * NV + a) * E + el], -gmj * stJ[((2 * N + i) * NV + a) * E + el]);
        double qz = fma(op.gp[k], jzp[a], -op.gm[k] * jzm[a]);
#pragma unroll
        for (int m = 0; m < N; ++m) {
          qx = fma(sD[i * N + m], (double)su[((j * N + m) * NV + a) * E], qx);
          qy = fma(sD[j * N + m], (double)su[((m * N + i) * NV + a) * E], qy);
          qz = fma(op.D[k * N + m], (double)sU[((size_t)(NFP * m + ij) * NV + a) * E + el], qz);
        }
        double q3[3];
        to_physical(S, rj, qx, qy, qz, q3);
#pragma unroll
        for (int n = 0; n < 3; ++n) {
          sQ[((n * NV + a) * NFP + ij) * E + el] = q3[n];
          zm[n][a] = fma(op.lm[k], q3[n], zm[n][a]);
          zp[n][a] = fma(op.lp[k], q3[n], zp[n][a]);
        }
      }
    }
    __syncthreads();  // Q of the slice is complete; stage k&1 has been consumed
    if (tid == 0 && k + 2 < N) issue_stage(k & 1, k + 2);
    // x / y faces of the slice: 4 N flux points per element, one thread each
    for (int t = ij; t < 4 * N; t += NFP) {
      const int f = t / N, m = t % N;
      const int base = f < 2 ? m * N : m, stride = f < 2 ? 1 : N;
      const double *lc = sL + (f & 1) * N;
      const int fp = f * NFP + m + N * k;
      double nrm[3], uf[NV], qf[3][NV], G[NV];
#pragma unroll
      for (int n = 0; n < 3; ++n) nrm[n] = fp_n[((size_t)n * NF + fp) * ld + e];
      const int pe = BND ? fp_pe[(size_t)fp * ld + e] : 0;
#pragma unroll
      for (int a = 0; a < NV; ++a) uf[a] = 0.0;
#pragma unroll
      for (int n = 0; n < 3; ++n)
#pragma unroll
        for (int a = 0; a < NV; ++a) qf[n][a] = 0.0;
#pragma unroll
      for (int mm = 0; mm < N; ++mm) {
        const double l = lc[mm];
        const int pt = base + mm * stride;
#pragma unroll
        for (int a = 0; a < NV; ++a) uf[a] = fma(l, (double)su[(pt * NV + a) * E], uf[a]);
#pragma unroll
        for (int n = 0; n < 3; ++n)
#pragma unroll
          for (int a = 0; a < NV; ++a) qf[n][a] = fma(l, sQ[((n * NV + a) * NFP + pt) * E + el], qf[n][a]);
      }
      face_visc<BND>(uf, qf, nrm, ph, pe, bcs, G);
      if (act) {
#pragma unroll
        for (int a = 0; a < NV; ++a) gf[((size_t)fp * NV + a) * ld + e] = G[a];
      }
    }
    if (k + 1 < N) __syncthreads();  // before the next slice overwrites sQ
  }
  // z faces of the column
#pragma unroll
  for (int s = 0; s < 2; ++s) {
    const int fp = (4 + s) * NFP + ij;
    double nrm[3], uf[NV], G[NV];
#pragma unroll
    for (int n = 0; n < 3; ++n) nrm[n] = fp_n[((size_t)n * NF + fp) * ld + e];
    const int pe = BND ? fp_pe[(size_t)fp * ld + e] : 0;
#pragma unroll
    for (int a = 0; a < NV; ++a) uf[a] = 0.0;
#pragma unroll
    for (int m = 0; m < N; ++m)
#pragma unroll
      for (int a = 0; a < NV; ++a)
        uf[a] = fma(s ? op.lp[m] : op.lm[m], (double)sU[((size_t)(NFP * m + ij) * NV + a) * E + el], uf[a]);
    face_visc<BND>(uf, s ? zp : zm, nrm, ph, pe, bcs, G);
    if (act) {
#pragma unroll
      for (int a = 0; a < NV; ++a) gf[((size_t)fp * NV + a) * ld + e] = G[a];
    }
  }
}

// ---------------------------------------------------------------------------------------------
// host side: tensor maps and launches
// ---------------------------------------------------------------------------------------------
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

template <int N, int E>
struct Maps {
  CUtensorMap U, S, R, R1, J;
};

template <int N, int E, typename T>
bool make_maps(const DevConsts &c, const void *u, const double *jump, Maps<N, E> &m, bool need_j) {
  constexpr int NFP = N * N, NU = N * NFP;
  const uint64_t ld = (uint64_t)c.ld;
  bool ok = encode3(&m.U, sizeof(T) == 8, u, ld, NFP * NV, N, ld, (uint64_t)NFP * NV * ld, E, NFP * NV, N);
  ok = ok && encode3(&m.S, true, c.smat, ld, NU, 9, ld, (uint64_t)NU * ld, E, NFP, 9);
  ok = ok && encode3(&m.R, true, c.rcpj, ld, NFP, N, ld, (uint64_t)NFP * ld, E, NFP, N);
  ok = ok && encode3(&m.R1, true, c.rcpj, ld, NFP, N, ld, (uint64_t)NFP * ld, E, NFP, 1);
  if (need_j) ok = ok && encode3(&m.J, true, jump, ld, NFP * NV, 6, ld, (uint64_t)NFP * NV * ld, E, N * NV, 4);
  else m.J = m.R;
  return ok;
}

template <typename K>
cudaError_t set_smem(K kern, size_t smem, bool &done) {
  if (done) return cudaSuccess;
  cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
  done = e == cudaSuccess;
  return e;
}

template <int N, int E, bool NS, typename T, int CAP = 8>
cudaError_t launch_rhs(const DevConsts &c, const double *h_ops, const void *u, const double *jump, const double *dt, void *rhs,
                       cudaStream_t s) {
  constexpr int NB1 = 1;
  using L2 = RhsLay<N, E, NS, T, 2>;
  using L1 = RhsLay<N, E, NS, T, NB1>;
  // double-buffer F~ when that does not cost a resident CTA
  constexpr int NB = (L2::TOTAL <= SMEM_MAX && min_blocks(L2::TOTAL, N * N * E) == min_blocks(L1::TOTAL, N * N * E)) ? 2 : 1;
  using L = RhsLay<N, E, NS, T, NB>;
  static_assert(L::TOTAL <= SMEM_MAX, "shared memory");
  constexpr int MINB = min_blocks(L::TOTAL, N * N * E) < CAP ? min_blocks(L::TOTAL, N * N * E) : CAP;
  Maps<N, E> m;
  if (!make_maps<N, E, T>(c, u, jump, m, NS)) return cudaErrorNotSupported;
  auto kern = k_hex_rhs_tma<N, E, NS, T, NB, MINB>;
  static bool done = false;
  cudaError_t err = set_smem(kern, L::TOTAL, done);
  if (err != cudaSuccess) return err;
  const Ops1D<N> op = make_ops<N>(h_ops);
  kern<<<(unsigned)((c.Nel + E - 1) / E), N * N * E, L::TOTAL, s>>>(m.U, m.S, m.R, m.J, op, c.ph, jump, dt, (T *)rhs, c.ld, c.Nel);
  return cudaGetLastError();
}

template <int N, int E, typename T, int CAP = 8>
cudaError_t launch_gradface(const DevConsts &c, const double *h_ops, const void *u, const double *jump, double *gf, cudaStream_t s) {
  using L = GfLay<N, E, T>;
  static_assert(L::TOTAL <= SMEM_MAX, "shared memory");
  constexpr int MINB = min_blocks(L::TOTAL, N * N * E) < CAP ? min_blocks(L::TOTAL, N * N * E) : CAP;
  Maps<N, E> m;
  if (!make_maps<N, E, T>(c, u, jump, m, true)) return cudaErrorNotSupported;
  const Ops1D<N> op = make_ops<N>(h_ops);
  const unsigned grid = (unsigned)((c.Nel + E - 1) / E);
  cudaError_t err;
  if (c.nbnd) {
    auto kern = k_hex_gradface<N, E, true, T, MINB>;
    static bool done = false;
    if ((err = set_smem(kern, L::TOTAL, done)) != cudaSuccess) return err;
    kern<<<grid, N * N * E, L::TOTAL, s>>>(m.U, m.S, m.R1, m.J, op, c.ph, jump, c.fp_n, c.fp_pe, c.bcs, gf, c.ld, c.Nel);
  } else {
    auto kern = k_hex_gradface<N, E, false, T, MINB>;
    static bool done = false;
    if ((err = set_smem(kern, L::TOTAL, done)) != cudaSuccess) return err;
    kern<<<grid, N * N * E, L::TOTAL, s>>>(m.U, m.S, m.R1, m.J, op, c.ph, jump, c.fp_n, c.fp_pe, c.bcs, gf, c.ld, c.Nel);
  }
  return cudaGetLastError();
}

// elements per CTA for each n = p + 1 (row segments of E*8 bytes)
template <int N>
struct Cfg {
  static constexpr int E = N <= 2 ? 32 : (N == 3 ? 16 : 8);
};

template <int N, typename T>
constexpr bool fits() {
  return GfLay<N, Cfg<N>::E, T>::TOTAL <= SMEM_MAX && RhsLay<N, Cfg<N>::E, true, T, 1>::TOTAL <= SMEM_MAX && N * N * Cfg<N>::E <= 1024;
}

int env_e() {
  static const int v = getenv("FR_TMA_E") ? atoi(getenv("FR_TMA_E")) : 0;
  return v;
}

template <int N, typename T>
cudaError_t rhs_n(const DevConsts &c, const double *h_ops, const void *u, const double *jump, const double *dt, void *rhs, cudaStream_t s) {
  if constexpr (fits<N, T>()) {
    if constexpr (N == 5 && sizeof(T) == 8) {  // tuning variants (FR_TMA_E = 16 | 12 | 81 (E = 8, one CTA per SM))
      if (env_e() == 16) return c.ns ? launch_rhs<N, 16, true, T>(c, h_ops, u, jump, dt, rhs, s) : launch_rhs<N, 16, false, T>(c, h_ops, u, jump, dt, rhs, s);
      if (env_e() == 12) return c.ns ? launch_rhs<N, 12, true, T>(c, h_ops, u, jump, dt, rhs, s) : launch_rhs<N, 12, false, T>(c, h_ops, u, jump, dt, rhs, s);
      if (env_e() == 81) return c.ns ? launch_rhs<N, 8, true, T, 1>(c, h_ops, u, jump, dt, rhs, s) : launch_rhs<N, 8, false, T, 1>(c, h_ops, u, jump, dt, rhs, s);
    }
    constexpr int E = Cfg<N>::E;
    return c.ns ? launch_rhs<N, E, true, T>(c, h_ops, u, jump, dt, rhs, s) : launch_rhs<N, E, false, T>(c, h_ops, u, jump, dt, rhs, s);
  } else {
    return cudaErrorNotSupported;
  }
}

template <int N, typename T>
cudaError_t gradface_n(const DevConsts &c, const double *h_ops, const void *u, const double *jump, double *gf, cudaStream_t s) {
  if constexpr (fits<N, T>()) {
    if constexpr (N == 5 && sizeof(T) == 8) {
      if (env_e() == 16) return launch_gradface<N, 16, T>(c, h_ops, u, jump, gf, s);
      if (env_e() == 12) return launch_gradface<N, 12, T>(c, h_ops, u, jump, gf, s);
      if (env_e() == 81) return launch_gradface<N, 8, T, 1>(c, h_ops, u, jump, gf, s);
    }
    return launch_gradface<N, Cfg<N>::E, T>(c, h_ops, u, jump, gf, s);
  } else {
    return cudaErrorNotSupported;
  }
}

}  // namespace

bool hex_tma_supported(int n, bool f64) {
  if (getenv("FR_NO_TMA")) return false;
  if (!encoder()) return false;
  switch (n) {
#define FR_CASE(NN) case NN: return f64 ? fits<NN, double>() : fits<NN, float>();
    FR_CASE(2) FR_CASE(3) FR_CASE(4) FR_CASE(5) FR_CASE(6) FR_CASE(7)
#undef FR_CASE
    default: return false;
  }
}

cudaError_t hex_tma_rhs(const DevConsts &c, const double *h_ops, const void *u, const double *jump, const double *dt, void *rhs,
                        cudaStream_t s) {
  switch (c.n) {
#define FR_CASE(NN) case NN: return c.f64 ? rhs_n<NN, double>(c, h_ops, u, jump, dt, rhs, s) : rhs_n<NN, float>(c, h_ops, u, jump, dt, rhs, s);
    FR_CASE(2) FR_CASE(3) FR_CASE(4) FR_CASE(5) FR_CASE(6) FR_CASE(7)
#undef FR_CASE
    default: return cudaErrorNotSupported;
  }
}

cudaError_t hex_tma_gradface(const DevConsts &c, const double *h_ops, const void *u, const double *jump, double *gf, cudaStream_t s) {
  switch (c.n) {
#define FR_CASE(NN) case NN: return c.f64 ? gradface_n<NN, double>(c, h_ops, u, jump, gf, s) : gradface_n<NN, float>(c, h_ops, u, jump, gf, s);
    FR_CASE(2) FR_CASE(3) FR_CASE(4) FR_CASE(5) FR_CASE(6) FR_CASE(7)
#undef FR_CASE
    default: return cudaErrorNotSupported;
  }
}

}  // namespace fr
