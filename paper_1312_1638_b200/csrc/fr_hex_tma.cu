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
#include "fr_tma.cuh"

namespace fr {
namespace {

// ---------------------------------------------------------------------------------------------
// shared-memory layouts (byte offsets from a 128-byte aligned base)
// ---------------------------------------------------------------------------------------------
template <int N, int E, bool NS, typename T, int NB>
struct RhsLay {
  static constexpr int NFP = N * N, NU = N * NFP;
  static constexpr size_t BAR = 0;
  static constexpr size_t OPS = 128;  // sD, sDh, sGm, sGp
  static constexpr size_t U = OPS + al128((2 * N * N + 2 * N) * 8);
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
  static constexpr size_t OPS = 128;  // sD [N*N], sL [2][N], sGm [N], sGp [N]
  static constexpr size_t U = OPS + al128((N * N + 4 * N) * 8);
  static constexpr uint32_t U_TX = NU * NV * E * sizeof(T);
  static constexpr size_t JZ = U + al128(U_TX);                   // jumps of the two z faces [2][NFP*NV][E], loaded once
  static constexpr uint32_t JZ_TX = 2 * NFP * NV * E * 8;
  static constexpr size_t SS = JZ + al128(JZ_TX);                 // S of the current slice: ONE buffer, refilled during the face phase
  static constexpr uint32_t S_TX = 9 * NFP * E * 8, R_TX = NFP * E * 8, J_TX = 4 * N * NV * E * 8;
  static constexpr size_t ST = SS + al128(S_TX);                  // two stages of {1/J, x/y-face jumps}
  static constexpr size_t ST_J = al128(R_TX);
  static constexpr size_t ST_BYTES = ST_J + al128(J_TX);
  static constexpr size_t Q = ST + 2 * ST_BYTES;
  static constexpr size_t Q_BYTES = 3 * NV * NFP * E * 8;
  static constexpr size_t TOTAL = Q + Q_BYTES + 128;
};

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
  double *sD = (double *)(sm + L::OPS), *sDh = sD + N * N, *sGm = sDh + N * N, *sGp = sGm + N;
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
  for (int t = tid; t < N; t += NFP * E) { sGm[t] = op.gm[t]; sGp[t] = op.gp[t]; }
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
  // z-face jumps of this column: re-read from L2 in every slice, one variable ahead of their use, instead of
  // staying in registers (10 values) across the whole kernel.
  auto ldj = [&](int face, int a) { return ld_nc_once(jump + ((size_t)(face * NFP + ij) * NV + a) * ld + e); };
  double jzm[NV], jzp[NV];
  auto load_jz = [&]() {
#pragma unroll
    for (int a = 0; a < NV; ++a) { jzm[a] = ldj(4, a); jzp[a] = ldj(5, a); }
  };
  if (NS) load_jz();
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
    double *buf = sF + (NB == 2 ? (k & 1) : 0) * (2 * NV * NFP * E);
    {
      double S[3][3], uu[NV];
#pragma unroll
      for (int a = 0; a < 3; ++a)
#pragma unroll
        for (int b = 0; b < 3; ++b) S[a][b] = stS[((a * 3 + b) * NFP + ij) * E + el];
      const T *su = sU + (size_t)(NFP * k) * NV * E + el;  // slice k
#pragma unroll
      for (int a = 0; a < NV; ++a) uu[a] = (double)su[(ij * NV + a) * E];
      // primitive variables (Eq 20-21)
      const double rrho = 1.0 / uu[0], En = uu[4];
      double v[3], ke = 0;
#pragma unroll
      for (int d = 0; d < 3; ++d) { v[d] = uu[1 + d] * rrho; ke += uu[1 + d] * v[d]; }
      const double p = (ph.gamma - 1.0) * (En - 0.5 * ke);
      // viscous stress Tm and the energy flux w = v.Tm + (mu gamma / Pr) grad e  (Eq 22-24, A8), built variable by
      // variable from the corrected physical gradients so that the 15 gradient values are never all live
      double Tm[3][3], w[3];
      if (NS) {
        const double rj = sRJ[(NFP * k + ij) * E + el];
        const double gmi = sGm[i], gpi = sGp[i], gmj = sGm[j], gpj = sGp[j];
        double g0[3], dv[3][3], de[3];
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
          double g[3];
          to_physical(S, rj, qx, qy, qz, g);
#pragma unroll
          for (int n = 0; n < 3; ++n) {
            if (a == 0) g0[n] = g[n];
            else if (a < 4) dv[n][a - 1] = (g[n] - v[a - 1] * g0[n]) * rrho;   // d_n v_j by the quotient rule
            else de[n] = (g[n] - (En * rrho) * g0[n]) * rrho;
          }
        }
        const double lam = -2.0 / 3.0 * ph.mu * (dv[0][0] + dv[1][1] + dv[2][2]);
#pragma unroll
        for (int a = 0; a < 3; ++a)
#pragma unroll
          for (int b = 0; b < 3; ++b) Tm[a][b] = ph.mu * (dv[a][b] + dv[b][a]) + (a == b ? lam : 0.0);
        const double kap = ph.mu * ph.gamma / ph.Pr;
#pragma unroll
        for (int n = 0; n < 3; ++n) {
          double d = de[n], vt = 0;
#pragma unroll
          for (int b = 0; b < 3; ++b) { d -= v[b] * dv[n][b]; vt += v[b] * Tm[b][n]; }
          w[n] = vt + kap * d;
        }
      }
      if (NB == 1 && k > 0) __syncthreads();  // the previous slice's contraction has finished reading sF
      // F~_i = sum_n S[i][n] (f_inv - f_vis)_n  (Eq 12), one variable at a time: x/y parts to shared memory,
      // z part straight into the column accumulators
#pragma unroll
      for (int a = 0; a < NV; ++a) {
        double f[3];
#pragma unroll
        for (int n = 0; n < 3; ++n) {
          if (a == 0) f[n] = uu[1 + n];
          else if (a < 4) { f[n] = uu[1 + n] * v[a - 1] + (a - 1 == n ? p : 0.0); if (NS) f[n] -= Tm[n][a - 1]; }
          else { f[n] = v[n] * (En + p); if (NS) f[n] -= w[n]; }
        }
        buf[((0 * NV + a) * NFP + ij) * E + el] = fma(S[0][0], f[0], fma(S[0][1], f[1], S[0][2] * f[2]));
        buf[((1 * NV + a) * NFP + ij) * E + el] = fma(S[1][0], f[0], fma(S[1][1], f[1], S[1][2] * f[2]));
        const double fz = fma(S[2][0], f[0], fma(S[2][1], f[1], S[2][2] * f[2]));
#pragma unroll
        for (int kk = 0; kk < N; ++kk) acc[kk][a] = fma(op.Dh[kk * N + k], fz, acc[kk][a]);
      }
    }
    __syncthreads();
    // every thread has consumed stage k&1: refill it with slice k+2
    if (tid == 0 && k + 2 < N) issue_stage(k & 1, k + 2);
    if (NS && k + 1 < N) load_jz();
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
  const double gmi = sGm[i], gpi = sGp[i], gmj = sGm[j], gpj = sGp[j];
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
// tmU, tmS, tmJ as above; tmR: rcpj as (ld, NFP, N), box (E, NFP, 1).
// SQ: also store Q slice by slice (bulk tensor store of the shared-memory slice) for k_hex_fluxdiv_tma;
// tmQ: Q workspace as (ld, NV*NFP, 3N), box (E, NV*NFP, 3): slice k, component n, variable a, point ij.
template <int N, int E, bool BND, bool SQ, typename T, int MINB>
__global__ void __launch_bounds__(N *N *E, MINB)
    k_hex_gradface(const __grid_constant__ CUtensorMap tmU, const __grid_constant__ CUtensorMap tmS,
                   const __grid_constant__ CUtensorMap tmR, const __grid_constant__ CUtensorMap tmJ,
                   const __grid_constant__ CUtensorMap tmQ, const __grid_constant__ CUtensorMap tmJz, Ops1D<N> op, Phys ph,
                   const double *__restrict__ jump, const double *__restrict__ fp_n, const int32_t *__restrict__ fp_pe,
                   const BcDev *__restrict__ bcs, double *__restrict__ gf, int64_t ld, int64_t Nel) {
  using L = GfLay<N, E, T>;
  constexpr int NFP = N * N, NF = 6 * NFP;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  unsigned char *sm = smem_raw + ((128u - (smem_addr(smem_raw) & 127u)) & 127u);  // stays in the shared address space
  uint64_t *bar = (uint64_t *)(sm + L::BAR);
  double *sD = (double *)(sm + L::OPS), *sL = sD + N * N;  // sL[0][m] = l_m(-1), sL[1][m] = l_m(+1)
  double *sGm = sL + 2 * N, *sGp = sGm + N;
  const T *sU = (const T *)(sm + L::U);
  const double *sJz = (const double *)(sm + L::JZ);
  const double *stS = (const double *)(sm + L::SS);
  unsigned char *sSt = sm + L::ST;
  double *sQ = (double *)(sm + L::Q);  // [3][NFP][NV][E]
  const int tid = threadIdx.x, el = tid % E, ij = tid / E, i = ij % N, j = ij / N;
  const int e0 = blockIdx.x * E;
  const int64_t e = (int64_t)e0 + el;
  const bool act = e < Nel;

  if (tid == 0) {
    mbar_init(&bar[0], 1); mbar_init(&bar[1], 1); mbar_init(&bar[2], 1); mbar_init(&bar[3], 1);
    fence_barrier_init();
    fence_proxy_async();
  }
  for (int t = tid; t < N * N; t += NFP * E) sD[t] = op.D[t];
  for (int t = tid; t < N; t += NFP * E) { sL[t] = op.lm[t]; sL[N + t] = op.lp[t]; sGm[t] = op.gm[t]; sGp[t] = op.gp[t]; }
  __syncthreads();
  auto issue_stage = [&](int s, int k) {
    mbar_expect_tx(&bar[1 + s], L::R_TX + L::J_TX);
    tma_load_3d(sSt + s * L::ST_BYTES, &tmR, e0, 0, k, &bar[1 + s]);
    tma_load_3d(sSt + s * L::ST_BYTES + L::ST_J, &tmJ, e0, N * k * NV, 0, &bar[1 + s]);
  };
  auto issue_S = [&](int k) {
    mbar_expect_tx(&bar[3], L::S_TX);
    tma_load_3d(sm + L::SS, &tmS, e0, NFP * k, 0, &bar[3]);
  };
  if (tid == 0) {
    mbar_expect_tx(&bar[0], L::U_TX + L::JZ_TX);
    tma_load_3d(sm + L::U, &tmU, e0, 0, 0, &bar[0]);
    tma_load_3d(sm + L::JZ, &tmJz, e0, 0, 4, &bar[0]);
    issue_S(0);
    issue_stage(0, 0);
    if (N > 1) issue_stage(1, 1);
  }
  double zm[3][NV], zp[3][NV];  // Q interpolated to the two z faces of this column
#pragma unroll
  for (int n = 0; n < 3; ++n)
#pragma unroll
    for (int a = 0; a < NV; ++a) zm[n][a] = zp[n][a] = 0.0;
  mbar_wait(&bar[0], 0);

#pragma unroll
  for (int k = 0; k < N; ++k) {
    mbar_wait(&bar[1 + (k & 1)], (k >> 1) & 1);
    mbar_wait(&bar[3], k & 1);
    const double *stR = (const double *)(sSt + (k & 1) * L::ST_BYTES);
    const double *stJ = (const double *)(sSt + (k & 1) * L::ST_BYTES + L::ST_J);
    const T *su = sU + (size_t)(NFP * k) * NV * E + el;  // slice k
    {
      double S[3][3];
#pragma unroll
      for (int a = 0; a < 3; ++a)
#pragma unroll
        for (int b = 0; b < 3; ++b) S[a][b] = stS[((a * 3 + b) * NFP + ij) * E + el];
      const double rj = stR[ij * E + el];
      const double gmi = sGm[i], gpi = sGp[i], gmj = sGm[j], gpj = sGp[j];
#pragma unroll
      for (int a = 0; a < NV; ++a) {
        double qx = fma(gpi, stJ[((1 * N + j) * NV + a) * E + el], -gmi * stJ[((0 * N + j) * NV + a) * E + el]);
        double qy = fma(gpj, stJ[((3 * N + i) * NV + a) * E + el], -gmj * stJ[((2 * N + i) * NV + a) * E + el]);
        double qz = fma(op.gp[k], sJz[((1 * NFP + ij) * NV + a) * E + el], -op.gm[k] * sJz[((0 * NFP + ij) * NV + a) * E + el]);
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
          sQ[((n * NFP + ij) * NV + a) * E + el] = q3[n];
          zm[n][a] = fma(op.lm[k], q3[n], zm[n][a]);
          zp[n][a] = fma(op.lp[k], q3[n], zp[n][a]);
        }
      }
    }
    if (SQ) fence_proxy_async();  // make the sQ writes visible to the bulk store
    __syncthreads();  // Q of the slice is complete; stage k&1 has been consumed
    if (tid == 0 && k + 1 < N) issue_S(k + 1);
    if (tid == 0 && k + 2 < N) issue_stage(k & 1, k + 2);
    if (SQ && tid == 0) { tma_store_3d(&tmQ, e0, 0, 3 * k, sQ); tma_store_commit(); }
    // x / y faces of the slice: 4 N flux points per element, one thread each
    for (int t = ij; t < 4 * N; t += NFP) {
      const int f = t / N, m = t % N;
      const int base = f < 2 ? m * N : m, stride = f < 2 ? 1 : N;
      const double *lc = sL + (f & 1) * N;
      const int fp = f * NFP + m + N * k;
      double nrm[3], uf[NV], G[NV];
#pragma unroll
      for (int n = 0; n < 3; ++n) nrm[n] = fp_n[((size_t)n * NF + fp) * ld + e];
#pragma unroll
      for (int a = 0; a < NV; ++a) uf[a] = 0.0;
#pragma unroll
      for (int mm = 0; mm < N; ++mm) {
        const double l = lc[mm];
#pragma unroll
        for (int a = 0; a < NV; ++a) uf[a] = fma(l, (double)su[((base + mm * stride) * NV + a) * E], uf[a]);
      }
      if constexpr (BND) {
        const int pe = fp_pe[(size_t)fp * ld + e];
        double qf[3][NV];
#pragma unroll
        for (int n = 0; n < 3; ++n)
#pragma unroll
          for (int a = 0; a < NV; ++a) {
            double q = 0;
#pragma unroll
            for (int mm = 0; mm < N; ++mm) q = fma(lc[mm], sQ[((n * NFP + base + mm * stride) * NV + a) * E + el], q);
            qf[n][a] = q;
          }
        face_visc<BND>(uf, qf, nrm, ph, pe, bcs, G);
      } else {
        visc_normal_stream(uf, nrm, ph, [&](int a, double *g) {
#pragma unroll
          for (int n = 0; n < 3; ++n) {
            double q = 0;
#pragma unroll
            for (int mm = 0; mm < N; ++mm) q = fma(lc[mm], sQ[((n * NFP + base + mm * stride) * NV + a) * E + el], q);
            g[n] = q;
          }
        }, G);
      }
      if (act) {
#pragma unroll
        for (int a = 0; a < NV; ++a) gf[((size_t)fp * NV + a) * ld + e] = G[a];
      }
    }
    if (SQ && tid == 0) tma_store_wait_read();  // the bulk store has read sQ
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
    if constexpr (BND) face_visc<BND>(uf, s ? zp : zm, nrm, ph, pe, bcs, G);
    else visc_normal_stream(uf, nrm, ph, [&](int a, double *g) {
#pragma unroll
      for (int n = 0; n < 3; ++n) g[n] = s ? zp[n][a] : zm[n][a];
    }, G);
    if (act) {
#pragma unroll
      for (int a = 0; a < NV; ++a) gf[((size_t)fp * NV + a) * ld + e] = G[a];
    }
  }
}

// ---------------------------------------------------------------------------------------------
// host side: tensor maps and launches
// ---------------------------------------------------------------------------------------------
template <int N, int E>
struct Maps {
  CUtensorMap U, S, R, R1, J, Jz, Q;
};

template <int N, int E, typename T>
bool make_maps(const DevConsts &c, const void *u, const double *jump, Maps<N, E> &m, bool need_j, const double *q = nullptr) {
  constexpr int NFP = N * N, NU = N * NFP;
  const uint64_t ld = (uint64_t)c.ld;
  bool ok = encode3(&m.U, sizeof(T) == 8, u, ld, NFP * NV, N, ld, (uint64_t)NFP * NV * ld, E, NFP * NV, N);
  ok = ok && encode3(&m.S, true, c.smat, ld, NU, 9, ld, (uint64_t)NU * ld, E, NFP, 9);
  ok = ok && encode3(&m.R, true, c.rcpj, ld, NFP, N, ld, (uint64_t)NFP * ld, E, NFP, N);
  ok = ok && encode3(&m.R1, true, c.rcpj, ld, NFP, N, ld, (uint64_t)NFP * ld, E, NFP, 1);
  if (need_j) {
    ok = ok && encode3(&m.J, true, jump, ld, NFP * NV, 6, ld, (uint64_t)NFP * NV * ld, E, N * NV, 4);
    ok = ok && encode3(&m.Jz, true, jump, ld, NFP * NV, 6, ld, (uint64_t)NFP * NV * ld, E, NFP * NV, 2);
  } else {
    m.J = m.R; m.Jz = m.R;
  }
  if (q) ok = ok && encode3(&m.Q, true, q, ld, NV * NFP, 3 * N, ld, (uint64_t)NV * NFP * ld, E, NV * NFP, 3);
  else m.Q = m.R;
  return ok;
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

template <int N, int E, bool BND, bool SQ, typename T, int MINB>
cudaError_t launch_gradface_k(const DevConsts &c, const Maps<N, E> &m, const Ops1D<N> &op, const double *jump, double *gf, cudaStream_t s) {
  using L = GfLay<N, E, T>;
  auto kern = k_hex_gradface<N, E, BND, SQ, T, MINB>;
  static bool done = false;
  cudaError_t err = set_smem(kern, L::TOTAL, done);
  if (err != cudaSuccess) return err;
  kern<<<(unsigned)((c.Nel + E - 1) / E), N * N * E, L::TOTAL, s>>>(m.U, m.S, m.R1, m.J, m.Q, m.Jz, op, c.ph, jump, c.fp_n, c.fp_pe, c.bcs, gf,
                                                                  c.ld,
                                                                  c.Nel);
  return cudaGetLastError();
}

template <int N, int E, typename T, int CAP = 8>
cudaError_t launch_gradface(const DevConsts &c, const double *h_ops, const void *u, const double *jump, double *gf, double *q,
                            cudaStream_t s) {
  using L = GfLay<N, E, T>;
  static_assert(L::TOTAL <= SMEM_MAX, "shared memory");
  constexpr int MINB = min_blocks(L::TOTAL, N * N * E) < CAP ? min_blocks(L::TOTAL, N * N * E) : CAP;
  Maps<N, E> m;
  if (!make_maps<N, E, T>(c, u, jump, m, true, q)) return cudaErrorNotSupported;
  const Ops1D<N> op = make_ops<N>(h_ops);
  if (c.nbnd) return q ? launch_gradface_k<N, E, true, true, T, MINB>(c, m, op, jump, gf, s) : launch_gradface_k<N, E, true, false, T, MINB>(c, m, op, jump, gf, s);
  return q ? launch_gradface_k<N, E, false, true, T, MINB>(c, m, op, jump, gf, s) : launch_gradface_k<N, E, false, false, T, MINB>(c, m, op, jump, gf, s);
}

template <int N, typename T>
constexpr bool fits() {
  return GfLay<N, Cfg<N>::E, T>::TOTAL <= SMEM_MAX && RhsLay<N, Cfg<N>::E, true, T, 1>::TOTAL <= SMEM_MAX && N * N * Cfg<N>::E <= 1024;
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
cudaError_t gradface_n(const DevConsts &c, const double *h_ops, const void *u, const double *jump, double *gf, double *q, cudaStream_t s) {
  if constexpr (fits<N, T>()) {
    if constexpr (N == 5 && sizeof(T) == 8) {
      if (env_e() == 16) return launch_gradface<N, 16, T>(c, h_ops, u, jump, gf, q, s);
      if (env_e() == 12) return launch_gradface<N, 12, T>(c, h_ops, u, jump, gf, q, s);
      if (env_e() == 81) return launch_gradface<N, 8, T, 1>(c, h_ops, u, jump, gf, q, s);
      if (env_e() == 4) return launch_gradface<N, 4, T>(c, h_ops, u, jump, gf, q, s);
    }
    return launch_gradface<N, Cfg<N>::E, T>(c, h_ops, u, jump, gf, q, s);
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

cudaError_t hex_tma_gradface(const DevConsts &c, const double *h_ops, const void *u, const double *jump, double *gf, double *q,
                             cudaStream_t s) {
  switch (c.n) {
#define FR_CASE(NN) case NN: return c.f64 ? gradface_n<NN, double>(c, h_ops, u, jump, gf, q, s) : gradface_n<NN, float>(c, h_ops, u, jump, gf, q, s);
    FR_CASE(2) FR_CASE(3) FR_CASE(4) FR_CASE(5) FR_CASE(6) FR_CASE(7)
#undef FR_CASE
    default: return cudaErrorNotSupported;
  }
}

}  // namespace fr
