// k_hex_fluxdiv_tma: parts (4), (6), (7) of the right-hand side on hexahedra in one TMA-pipelined kernel (sm_100a):
//   F~ = S f(U, Q)  (Eq 12 :214 with Eq 20-24),  R = -(1/J) {(M1 - M3 M2) F~ + M3 D~}  (Eq 18-19 / Eq 44 :772).
// A CTA owns E consecutive elements and walks them slice by slice (z = k).  Everything a slice needs -- the metric
// terms S (9 rows per point), the U slice and, for Navier-Stokes, the Q slice written by k_hex_gradface -- arrives
// in a two-stage ring of TMA box loads completing on mbarriers, issued two slices ahead by one thread.  F~ never
// leaves the SM: its x/y parts go through one shared-memory slice, its z part straight into the column accumulators.
#include "fr_tma.cuh"

namespace fr {
namespace {

// AFF: affine mesh (one set of metric terms per element, fr_api.cu): S and 1/J are read once per thread from the per-element
// tables and the ring carries no metric slice.  Euler: the ring holds the U slice only and ALL of D~ has a buffer of its own
// that is loaded at kernel start (EPI_ALL).
template <int N, int E, bool NS, typename T, int NB, bool AFF = false>
struct FdLay {
  static constexpr int NFP = N * N, NU = N * NFP;
  static constexpr size_t BAR = 0;
  static constexpr size_t OPS = 128;  // sDh [N*N], sGm [N], sGp [N]
  static constexpr size_t ST = OPS + al128((N * N + 2 * N) * 8);  // (sized for double operators)
  static constexpr uint32_t S_TX = AFF ? 0 : 9 * NFP * E * sizeof(T), U_TX = NFP * NV * E * sizeof(T), Q_TX = NS ? 3 * NV * NFP * E * sizeof(T) : 0;
  static constexpr size_t ST_U = al128(S_TX);
  static constexpr size_t ST_Q = ST_U + al128(U_TX);
  static constexpr size_t ST_BYTES = ST_Q + al128(Q_TX);
  static constexpr size_t F = ST + 2 * ST_BYTES;
  static constexpr size_t F_BYTES = 2 * NV * NFP * E * 8;
  // epilogue operands by TMA: D~ of the x/y faces, 1/J, D~ of the z faces.  EPI_ST: all into the stage buffers once they
  // are free (Navier-Stokes: the stages are large).  EPI_DED: the stages are too small for D~ of the x/y faces (Euler), which
  // gets a buffer of its own, loaded at kernel start; 1/J and the z faces still reuse the freed stages.
  static constexpr uint32_t DXY_TX = 4 * NFP * NV * E * sizeof(T), RJ_TX = NU * E * sizeof(T), DZ_TX = 2 * NFP * NV * E * sizeof(T);
  static constexpr size_t EP_RJ = al128(DXY_TX);
  static constexpr bool EPI_ALL = AFF && !NS && N >= 2;
  static constexpr uint32_t RJ_NEED = AFF ? 0 : RJ_TX;  // AFF: 1/J is one value per element, read from its table
  static constexpr bool EPI_ST = !EPI_ALL && N >= 2 && EP_RJ + RJ_NEED <= ST_BYTES && DZ_TX <= ST_BYTES;
  static constexpr bool EPI_DED = !EPI_ALL && N >= 2 && !EPI_ST && RJ_NEED <= ST_BYTES && DZ_TX <= ST_BYTES;
  static constexpr bool EPI_TMA = EPI_ST || EPI_DED;
  static constexpr size_t DED = F + al128(NB * F_BYTES);  // TMA destination: 128-byte aligned
  static constexpr size_t DED_Z = DED + al128(DXY_TX);     // EPI_ALL: D~ of the z faces behind D~ of the x/y faces
  static constexpr size_t TOTAL = DED + (EPI_DED ? al128(DXY_TX) : 0) + (EPI_ALL ? al128(DXY_TX) + al128(DZ_TX) : 0) + 128;  // + slack for the manual 128-byte alignment
};

// tmS: smat as (ld, NU, 9), box (E, NFP, 9);  tmU: u as (ld, NFP*NV, N), box (E, NFP*NV, 1);
// tmQ: Q workspace as (ld, NV*NFP, 3N), box (E, NV*NFP, 3)  (slice-major layout written by k_hex_gradface).
// Epilogue operands (when they fit the stage buffers): tmD4 / tmD2: D~ as (ld, NFP*NV, 6), boxes (E, NFP*NV, 4) / (E, NFP*NV, 2);
// tmR: rcpj as (ld, NFP, N), box (E, NFP, N).
template <int N, int E, bool NS, typename T, int NB, int MINB, bool AFF>
__global__ void __launch_bounds__(N *N *E, MINB)
    k_hex_fluxdiv_tma(const __grid_constant__ CUtensorMap tmS, const __grid_constant__ CUtensorMap tmU,
                      const __grid_constant__ CUtensorMap tmQ, const __grid_constant__ CUtensorMap tmD4,
                      const __grid_constant__ CUtensorMap tmD2, const __grid_constant__ CUtensorMap tmR, Ops1D<N> op, Phys ph,
                      const T *__restrict__ rcpj, const T *__restrict__ smat, bool aff, const T *__restrict__ dt, T *__restrict__ rhs,
                      int64_t ld, int64_t Nel) {
  using L = FdLay<N, E, NS, T, NB, AFF>;
  constexpr int NFP = N * N;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  unsigned char *sm = smem_raw + ((128u - (smem_addr(smem_raw) & 127u)) & 127u);  // stays in the shared address space
  uint64_t *bar = (uint64_t *)(sm + L::BAR);
  // Arithmetic in double in both storage precisions (the inviscid flux and its divergence are where cancellation happens).
  // Contractions in float were measured in single precision: no gain (0.192 ms either way on C3) and twice the freestream residual.
  using R = double;
  R *sDh = (R *)(sm + L::OPS), *sGm = sDh + N * N, *sGp = sGm + N;
  unsigned char *sSt = sm + L::ST;
  R *sF = (R *)(sm + L::F);  // [NB][2][NV][NFP][E]
  const int tid = threadIdx.x, el = tid % E, ij = patch_ij<N>(tid / E), i = ij % N, j = ij / N;  // 2 x 2 patches per warp (fr_tma.cuh)
  const int e0 = blockIdx.x * E, l0 = e0 % FR_BLK, eb = e0 / FR_BLK;  // first element: lane and element block (fp_row)
  const int64_t e = (int64_t)e0 + el;
  const bool act = e < Nel;

  if (tid == 0) {
    mbar_init(&bar[0], 1); mbar_init(&bar[1], 1); mbar_init(&bar[2], 1); mbar_init(&bar[3], 1); mbar_init(&bar[4], 1);
    fence_barrier_init();
    fence_proxy_async();
  }
  for (int t = tid; t < N * N; t += NFP * E) sDh[t] = op.Dh[t];
  for (int t = tid; t < N; t += NFP * E) { sGm[t] = op.gm[t]; sGp[t] = op.gp[t]; }
  __syncthreads();
  auto issue_stage = [&](int s, int k) {
    mbar_expect_tx(&bar[s], L::S_TX + L::U_TX + L::Q_TX);
    if (!AFF) tma_load_4d(sSt + s * L::ST_BYTES, &tmS, l0, NFP * k, 0, eb, &bar[s]);
    tma_load_3d(sSt + s * L::ST_BYTES + L::ST_U, &tmU, e0, 0, k, &bar[s]);
    if (NS) tma_load_4d(sSt + s * L::ST_BYTES + L::ST_Q, &tmQ, l0, 0, 3 * k, eb, &bar[s]);
  };
  if (tid == 0) {
    issue_stage(0, 0);
    if (N > 1) issue_stage(1, 1);
    if (L::EPI_DED || L::EPI_ALL) { mbar_expect_tx(&bar[2], L::DXY_TX); tma_load_4d(sm + L::DED, &tmD4, l0, 0, 0, eb, &bar[2]); }
    if (L::EPI_ALL) { mbar_expect_tx(&bar[3], L::DZ_TX); tma_load_4d(sm + L::DED_Z, &tmD2, l0, 0, 4, eb, &bar[3]); }
  }
  double Sr[3][3];  // AFF: the element's metric terms, [block][9][FR_BLK] (fr_api.cu)
  if (AFF) {
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
      for (int b = 0; b < 3; ++b) Sr[a][b] = (double)smat[((size_t)eb * 9 + a * 3 + b) * FR_BLK + l0 + el];
  }
  R acc[N][NV];
#pragma unroll
  for (int k = 0; k < N; ++k)
#pragma unroll
    for (int a = 0; a < NV; ++a) acc[k][a] = 0;

#pragma unroll
  for (int k = 0; k < N; ++k) {
    mbar_wait(&bar[k & 1], (k >> 1) & 1);
    const T *stS = (const T *)(sSt + (k & 1) * L::ST_BYTES);
    const T *stU = (const T *)(sSt + (k & 1) * L::ST_BYTES + L::ST_U);
    const T *stQ = (const T *)(sSt + (k & 1) * L::ST_BYTES + L::ST_Q);
    R *buf = sF + (NB == 2 ? (k & 1) : 0) * (2 * NV * NFP * E);
    {
      double S[3][3], uu[NV];
#pragma unroll
      for (int a = 0; a < 3; ++a)
#pragma unroll
        for (int b = 0; b < 3; ++b) S[a][b] = AFF ? Sr[a][b] : (double)stS[((a * 3 + b) * NFP + ij) * E + el];
#pragma unroll
      for (int a = 0; a < NV; ++a) uu[a] = (double)stU[(ij * NV + a) * E + el];
      // primitive variables (Eq 20-21) through the perturbation variables w about the reference state (fr_physics.cuh):
      // v = v0 + w_m / rho,  pp = p - p0;  with no reference state w = u and pp = p
      const double rrho = 1.0 / uu[0];
      double ww[NV], v[3], dvl[3], ke = 0, vw = 0;
      to_pert<3>(ph, uu, ww);
      const double Es = (ww[4] - ph.p0) * rrho;
#pragma unroll
      for (int d = 0; d < 3; ++d) {
        dvl[d] = ww[1 + d] * rrho;
        v[d] = ph.v0[d] + dvl[d];
        ke += ww[1 + d] * dvl[d];
        vw += ph.v0[d] * ww[1 + d];
      }
      const double pp = (ph.gamma - 1.0) * (fma(ph.hs0, ww[0], ww[4]) - vw - 0.5 * ke);
      // viscous stress Tm and energy flux w = v.Tm + (mu gamma / Pr) grad e  (Eq 22-24, A8), built variable by variable from
      // the gradient of the perturbation variables (formulas of subtract_viscous_flux, fr_physics.cuh)
      double Tm[3][3], w[3];
      if (NS) {
        double g0[3], dv[3][3], de[3];
#pragma unroll
        for (int a = 0; a < NV; ++a)
#pragma unroll
          for (int n = 0; n < 3; ++n) {
            const double g = (double)stQ[((n * NFP + ij) * NV + a) * E + el];
            if (a == 0) g0[n] = g;
            else if (a < 4) dv[n][a - 1] = (g - dvl[a - 1] * g0[n]) * rrho;  // d_n v_j by the quotient rule (Q = grad w)
            else de[n] = (g - Es * g0[n]) * rrho;
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
      // F~_i = sum_n S[i][n] (g_inv - f_vis)_n  (Eq 12; g = the inviscid flux in perturbation form), one variable at a time
#pragma unroll
      for (int a = 0; a < NV; ++a) {
        double f[3];
#pragma unroll
        for (int n = 0; n < 3; ++n) {
          if (a == 0) f[n] = fma(ph.v0[n], ww[0], ww[1 + n]);
          else if (a < 4) { f[n] = v[n] * ww[a] + (a - 1 == n ? pp : 0.0); if (NS) f[n] -= Tm[n][a - 1]; }
          else { f[n] = v[n] * (ww[4] + pp); if (NS) f[n] -= w[n]; }
        }
        buf[((0 * NV + a) * NFP + ij) * E + el] = (R)fma(S[0][0], f[0], fma(S[0][1], f[1], S[0][2] * f[2]));
        buf[((1 * NV + a) * NFP + ij) * E + el] = (R)fma(S[1][0], f[0], fma(S[1][1], f[1], S[1][2] * f[2]));
        const R fz = (R)fma(S[2][0], f[0], fma(S[2][1], f[1], S[2][2] * f[2]));
#pragma unroll
        for (int kk = 0; kk < N; ++kk) acc[kk][a] = fma(op.Dh[kk * N + k], fz, acc[kk][a]);
      }
    }
    fence_proxy_async();  // generic-proxy reads of the stage are ordered before the bulk copies that refill it (fr_hex_tma.cu, z faces)
    __syncthreads();
    // every thread has consumed stage k&1: refill it with slice k+2
    if (tid == 0 && k + 2 < N) issue_stage(k & 1, k + 2);
    if (L::EPI_ST && tid == 0 && k == N - 2) {  // this stage is not refilled any more: bring D~ (x/y faces) and 1/J
      mbar_expect_tx(&bar[2], L::DXY_TX);
      tma_load_4d(sSt + (k & 1) * L::ST_BYTES, &tmD4, l0, 0, 0, eb, &bar[2]);
      if (!AFF) {
        mbar_expect_tx(&bar[4], L::RJ_TX);
        tma_load_4d(sSt + (k & 1) * L::ST_BYTES + L::EP_RJ, &tmR, l0, 0, 0, eb, &bar[4]);
      }
    }
    if (L::EPI_DED && !AFF && tid == 0 && k == N - 2) {
      mbar_expect_tx(&bar[4], L::RJ_TX);
      tma_load_4d(sSt + (k & 1) * L::ST_BYTES, &tmR, l0, 0, 0, eb, &bar[4]);
    }
    if (L::EPI_TMA && tid == 0 && k == N - 1) {  // D~ of the z faces
      mbar_expect_tx(&bar[3], L::DZ_TX);
      tma_load_4d(sSt + (k & 1) * L::ST_BYTES, &tmD2, l0, 0, 4, eb, &bar[3]);
    }
    // x and y contractions within the slice
#pragma unroll
    for (int m = 0; m < N; ++m) {
      const R dx = sDh[i * N + m], dy = sDh[j * N + m];
#pragma unroll
      for (int a = 0; a < NV; ++a) {
        acc[k][a] = fma(dx, buf[((0 * NV + a) * NFP + j * N + m) * E + el], acc[k][a]);
        acc[k][a] = fma(dy, buf[((1 * NV + a) * NFP + m * N + i) * E + el], acc[k][a]);
      }
    }
  }
  // lifting M3 D~ and the -1/J scale (Eq 19); faces: 0,1 = x-,x+ (idx j + N k); 2,3 = y (i + N k); 4,5 = z (i + N j)
  const double gmi = (double)sGm[i], gpi = (double)sGp[i], gmj = (double)sGm[j], gpj = (double)sGp[j];
  if (L::EPI_TMA || L::EPI_ALL) {
    const T *sDxy = (const T *)((L::EPI_DED || L::EPI_ALL) ? sm + L::DED : sSt + ((N - 2) & 1) * L::ST_BYTES);  // [4][NFP*NV][E]
    const T *sRJ = (const T *)(sSt + ((N - 2) & 1) * L::ST_BYTES + (L::EPI_DED ? 0 : L::EP_RJ));  // [NU][E]
    const T *sDz = (const T *)(L::EPI_ALL ? sm + L::DED_Z : sSt + ((N - 1) & 1) * L::ST_BYTES);                // [2][NFP*NV][E]
    const double rj_el = AFF ? (double)rcpj[(size_t)eb * FR_BLK + l0 + el] : 0.0;  // [block][1][FR_BLK]
    mbar_wait(&bar[2], 0);
    mbar_wait(&bar[3], 0);
    if (!AFF) mbar_wait(&bar[4], 0);
    if (!act) return;
#pragma unroll
    for (int k = 0; k < N; ++k) {
      const int r = ij + NFP * k;
      const double rj = AFF ? rj_el : (double)sRJ[r * E + el];
      const int fx = j + N * k, fy = i + N * k;
      double r0 = 0;  // R~ of the mass equation: R_mj = R_wmj + v0_j R_wrho, R_E = R_wE + h0 R_wrho (fr_physics.cuh)
#pragma unroll
      for (int a = 0; a < NV; ++a) {
        double v = (double)acc[k][a];
        v = fma((double)op.gm[k], (double)sDz[((0 * NFP + ij) * NV + a) * E + el], v);
        v = fma((double)op.gp[k], (double)sDz[((1 * NFP + ij) * NV + a) * E + el], v);
        v = fma(gmi, (double)sDxy[((0 * NFP + fx) * NV + a) * E + el], v);
        v = fma(gpi, (double)sDxy[((1 * NFP + fx) * NV + a) * E + el], v);
        v = fma(gmj, (double)sDxy[((2 * NFP + fy) * NV + a) * E + el], v);
        v = fma(gpj, (double)sDxy[((3 * NFP + fy) * NV + a) * E + el], v);
        if (a == 0) r0 = v;
        else v = fma(a < 4 ? ph.v0[a - 1] : ph.h0, r0, v);
        rhs[((size_t)r * NV + a) * ld + e] = (T)(-v * rj);
      }
    }
    return;
  }
  if (!act) return;
  double dzm[NV], dzp[NV];
#pragma unroll
  for (int a = 0; a < NV; ++a) {
    dzm[a] = (double)dt[fp_row(true, ld, 6 * NFP * NV, (4 * NFP + ij) * NV + a, e)];
    dzp[a] = (double)dt[fp_row(true, ld, 6 * NFP * NV, (5 * NFP + ij) * NV + a, e)];
  }
#pragma unroll
  for (int k = 0; k < N; ++k) {
    const int r = ij + NFP * k;
    const double rj = (double)(aff ? rcpj[fp_row(true, ld, 1, 0, e)] : rcpj[fp_row(true, ld, N * NFP, r, e)]);
    const int fx = j + N * k, fy = i + N * k;
    double r0 = 0;
#pragma unroll
    for (int a = 0; a < NV; ++a) {
      double v = (double)acc[k][a];
      v = fma((double)op.gm[k], dzm[a], v);
      v = fma((double)op.gp[k], dzp[a], v);
      v = fma(gmi, (double)dt[fp_row(true, ld, 6 * NFP * NV, (0 * NFP + fx) * NV + a, e)], v);
      v = fma(gpi, (double)dt[fp_row(true, ld, 6 * NFP * NV, (1 * NFP + fx) * NV + a, e)], v);
      v = fma(gmj, (double)dt[fp_row(true, ld, 6 * NFP * NV, (2 * NFP + fy) * NV + a, e)], v);
      v = fma(gpj, (double)dt[fp_row(true, ld, 6 * NFP * NV, (3 * NFP + fy) * NV + a, e)], v);
      if (a == 0) r0 = v;
      else v = fma(a < 4 ? ph.v0[a - 1] : ph.h0, r0, v);
      rhs[((size_t)r * NV + a) * ld + e] = (T)(-v * rj);
    }
  }
}

template <int N, int E, bool NS, typename T, bool AFF>
cudaError_t launch_fluxdiv(const DevConsts &c, const double *h_ops, const void *u, const void *q, const void *dt, void *rhs,
                           cudaStream_t s) {
  constexpr int NFP = N * N, NU = N * NFP;
  using L2 = FdLay<N, E, NS, T, 2, AFF>;
  using L1 = FdLay<N, E, NS, T, 1, AFF>;
  // double-buffer F~ when that does not cost a resident CTA
  constexpr int REGS = 128;  // (96 registers for a third resident CTA: 176 bytes of spills at p = 4 in single precision, rejected)
  constexpr int NB = (L2::TOTAL <= SMEM_MAX && min_blocks(L2::TOTAL, N * N * E, REGS) == min_blocks(L1::TOTAL, N * N * E, REGS)) ? 2 : 1;
  using L = FdLay<N, E, NS, T, NB, AFF>;
  static_assert(L::TOTAL <= SMEM_MAX, "shared memory");
  constexpr int MINB = min_blocks(L::TOTAL, N * N * E, REGS);
  const uint64_t ld = (uint64_t)c.ld;
  static_assert(FR_BLK % E == 0, "a CTA's elements must lie in one element block");
  constexpr bool F64 = sizeof(T) == 8;
  bool fresh = true;
  MapCache::Ent *ent = ((MapCache *)c.map_cache)->get(NS ? 2 : 3, u, q, dt, fresh);
  CUtensorMap &mS = ent->m[0], &mU = ent->m[1], &mQ = ent->m[2], &mD4 = ent->m[3], &mD2 = ent->m[4], &mR = ent->m[5];
  bool ok = !fresh;
  if (fresh) {
  ok = encode_blk(&mS, F64, c.smat, ld, NU, 9, E, NFP, 9, c.aff ? 1 : 0);  // metric terms in T on this path (fr_api.cu)
  ok = ok && encode3(&mU, sizeof(T) == 8, u, ld, NFP * NV, N, ld, (uint64_t)NFP * NV * ld, E, NFP * NV, 1);  // caller layout
  if (NS) ok = ok && encode_blk(&mQ, F64, q, ld, NV * NFP, 3 * N, E, NV * NFP, 3);
  else mQ = mS;
  ok = ok && encode_blk(&mD4, F64, dt, ld, NFP * NV, 6, E, NFP * NV, 4);
  ok = ok && encode_blk(&mD2, F64, dt, ld, NFP * NV, 6, E, NFP * NV, 2);
  ok = ok && encode_blk(&mR, F64, c.rcpj, ld, NFP, N, E, NFP, N, c.aff ? 2 : 0);
  }
  if (!ok) { ent->id = -1; return cudaErrorNotSupported; }
  auto kern = k_hex_fluxdiv_tma<N, E, NS, T, NB, MINB, AFF>;
  static DevFlags done;
  cudaError_t err = set_smem(kern, L::TOTAL, done, c.dev);
  if (err != cudaSuccess) return err;
  const Ops1D<N> op = make_ops<N>(h_ops);
  kern<<<(unsigned)((c.Nel + E - 1) / E), N * N * E, L::TOTAL, s>>>(mS, mU, mQ, mD4, mD2, mR, op, c.ph, (const T *)c.rcpj, (const T *)c.smat, c.aff, (const T *)dt, (T *)rhs, c.ld,
                                                                  c.Nel);
  return cudaGetLastError();
}

template <int N, typename T>
constexpr bool fd_fits() {
  return FdLay<N, Cfg<N, T>::E_SLAB, true, T, 1>::TOTAL <= SMEM_MAX && N * N * Cfg<N, T>::E_SLAB <= 1024 && N * N * NV <= 256;
}

template <int N, typename T>
cudaError_t fluxdiv_n(const DevConsts &c, const double *h_ops, const void *u, const void *q, const void *dt, void *rhs, cudaStream_t s) {
  if constexpr (fd_fits<N, T>()) {
    constexpr int E = Cfg<N, T>::E_SLAB;
    if constexpr (FdLay<N, E, false, T, 1, true>::TOTAL <= SMEM_MAX && FdLay<N, E, true, T, 1, true>::EPI_TMA) {
      if (c.aff) return c.ns ? launch_fluxdiv<N, E, true, T, true>(c, h_ops, u, q, dt, rhs, s) : launch_fluxdiv<N, E, false, T, true>(c, h_ops, u, q, dt, rhs, s);
    }
    return c.ns ? launch_fluxdiv<N, E, true, T, false>(c, h_ops, u, q, dt, rhs, s) : launch_fluxdiv<N, E, false, T, false>(c, h_ops, u, q, dt, rhs, s);
  } else {
    return cudaErrorNotSupported;
  }
}

}  // namespace

bool hex_tma_fluxdiv_supported(int n, bool f64) {
  if (!encoder()) return false;
  switch (n) {
#define FR_CASE(NN) case NN: return f64 ? fd_fits<NN, double>() : fd_fits<NN, float>();
    FR_CASE(2) FR_CASE(3) FR_CASE(4) FR_CASE(5) FR_CASE(6) FR_CASE(7)
#undef FR_CASE
    default: return false;
  }
}

cudaError_t hex_tma_fluxdiv(const DevConsts &c, const double *h_ops, const void *u, const void *q, const void *dt, void *rhs,
                            cudaStream_t s) {
  switch (c.n) {
#define FR_CASE(NN) case NN: return c.f64 ? fluxdiv_n<NN, double>(c, h_ops, u, q, dt, rhs, s) : fluxdiv_n<NN, float>(c, h_ops, u, q, dt, rhs, s);
    FR_CASE(2) FR_CASE(3) FR_CASE(4) FR_CASE(5) FR_CASE(6) FR_CASE(7)
#undef FR_CASE
    default: return cudaErrorNotSupported;
  }
}

}  // namespace fr
