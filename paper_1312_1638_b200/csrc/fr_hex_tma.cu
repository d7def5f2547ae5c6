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
//   (k_hex_fluxdiv_tma, fr_hex_fluxdiv_tma.cu: F~ = S f(U, Q), R = -(1/J) {(M1 - M3 M2) F~ + M3 D~}.)
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
                   const uint8_t *__restrict__ face_need, const BcDev *__restrict__ bcs, double *__restrict__ gf, int64_t ld,
                   int64_t Nel) {
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
  const int e0 = blockIdx.x * E, l0 = e0 % FR_BLK, eb = e0 / FR_BLK;  // first element: lane and element block (fp_row)
  const int64_t e = (int64_t)e0 + el;
  const bool act = e < Nel;

  if (tid == 0) {
    mbar_init(&bar[0], 1); mbar_init(&bar[1], 1); mbar_init(&bar[2], 1); mbar_init(&bar[3], 1);
    mbar_init(&bar[4], 1); mbar_init(&bar[5], 1);  // second pass over the Q slices (z faces)
    fence_barrier_init();
    fence_proxy_async();
  }
  for (int t = tid; t < N * N; t += NFP * E) sD[t] = op.D[t];
  for (int t = tid; t < N; t += NFP * E) { sL[t] = op.lm[t]; sL[N + t] = op.lp[t]; sGm[t] = op.gm[t]; sGp[t] = op.gp[t]; }
  __syncthreads();
  auto issue_stage = [&](int s, int k) {
    mbar_expect_tx(&bar[1 + s], L::R_TX + L::J_TX);
    tma_load_4d(sSt + s * L::ST_BYTES, &tmR, l0, 0, k, eb, &bar[1 + s]);
    tma_load_4d(sSt + s * L::ST_BYTES + L::ST_J, &tmJ, l0, N * k * NV, 0, eb, &bar[1 + s]);
  };
  auto issue_S = [&](int k) {
    mbar_expect_tx(&bar[3], L::S_TX);
    tma_load_4d(sm + L::SS, &tmS, l0, NFP * k, 0, eb, &bar[3]);
  };
  if (tid == 0) {
    mbar_expect_tx(&bar[0], L::U_TX + L::JZ_TX);
    tma_load_3d(sm + L::U, &tmU, e0, 0, 0, &bar[0]);
    tma_load_4d(sm + L::JZ, &tmJz, l0, 0, 4, eb, &bar[0]);
    issue_S(0);
    issue_stage(0, 0);
    if (N > 1) issue_stage(1, 1);
  }
  // G^f of a face is needed only if its LDG weight (1/2 + beta on L sides, 1/2 - beta on R sides, Eq 27) is non-zero or it
  // lies on a boundary: with the paper's beta = 1/2 half of the faces are skipped.  x/y tasks visit the +1 faces first
  // (the L sides of structured meshes) so that skipped tasks fall into the same warps.
  constexpr int TPT = (4 * N + NFP - 1) / NFP;  // x/y-face tasks of a thread per slice
  bool need_xy[TPT];
#pragma unroll
  for (int q = 0; q < TPT; ++q) {
    const int t = ij + q * NFP;
    need_xy[q] = t < 4 * N && act && face_need[(size_t)(t < 2 * N ? 2 * (t / N) + 1 : 2 * (t / N - 2)) * ld + e] != 0;
  }
  const bool need_z[2] = {act && face_need[(size_t)4 * ld + e] != 0, act && face_need[(size_t)5 * ld + e] != 0};
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
        }
      }
    }
    if (SQ) fence_proxy_async();  // make the sQ writes visible to the bulk store
    __syncthreads();  // Q of the slice is complete; stage k&1 has been consumed
    if (tid == 0 && k + 1 < N) issue_S(k + 1);
    if (tid == 0 && k + 2 < N) issue_stage(k & 1, k + 2);
    if (SQ && tid == 0) { tma_store_4d(&tmQ, l0, 0, 3 * k, eb, sQ); tma_store_commit(); }
    // x / y faces of the slice: 4 N flux points per element, one thread each
#pragma unroll
    for (int q = 0; q < TPT; ++q) {
      if (!need_xy[q]) continue;
      const int t = ij + q * NFP;
      const int f = t < 2 * N ? 2 * (t / N) + 1 : 2 * (t / N - 2), m = t % N;  // faces 1, 3 (+x, +y), then 0, 2
      const int base = f < 2 ? m * N : m, stride = f < 2 ? 1 : N;
      const double *lc = sL + (f & 1) * N;
      const int fp = f * NFP + m + N * k;
      double nrm[3], uf[NV], G[NV];
#pragma unroll
      for (int n = 0; n < 3; ++n) nrm[n] = fp_n[fp_row(true, ld, 3 * NF, n * NF + fp, e)];
#pragma unroll
      for (int a = 0; a < NV; ++a) uf[a] = 0.0;
#pragma unroll
      for (int mm = 0; mm < N; ++mm) {
        const double l = lc[mm];
#pragma unroll
        for (int a = 0; a < NV; ++a) uf[a] = fma(l, (double)su[((base + mm * stride) * NV + a) * E], uf[a]);
      }
      if constexpr (BND) {
        const int pe = fp_pe[fp_row(true, ld, NF, fp, e)];
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
        for (int a = 0; a < NV; ++a) gf[fp_row(true, ld, NF * NV, fp * NV + a, e)] = G[a];
      }
    }
    if (SQ && tid == 0) tma_store_wait_read();  // the bulk store has read sQ
    if (k + 1 < N) __syncthreads();  // before the next slice overwrites sQ
  }
  // ---- z faces.  Q^f on them is sum_k l(+-1)_k Q(i, j, k): instead of carrying 2 x 15 accumulators through the slice
  // loop, the Q slices just stored are streamed once more (TMA loads, L2 hits) through two buffers that the slice loop
  // no longer needs: [SS .. Q) (S, 1/J, x/y jumps) and [U .. SS) (U block, z jumps).  The last slice is still in sQ.
  static_assert(L::Q - L::SS >= L::Q_BYTES && L::SS - L::U >= L::Q_BYTES, "Q slice does not fit the reused buffers");
  double ufz[2][NV];
#pragma unroll
  for (int s = 0; s < 2; ++s)
#pragma unroll
    for (int a = 0; a < NV; ++a) ufz[s][a] = 0.0;
#pragma unroll
  for (int m = 0; m < N; ++m)
#pragma unroll
    for (int a = 0; a < NV; ++a) {
      const double v = (double)sU[((size_t)(NFP * m + ij) * NV + a) * E + el];
      ufz[0][a] = fma(op.lm[m], v, ufz[0][a]);
      ufz[1][a] = fma(op.lp[m], v, ufz[1][a]);
    }
  __syncthreads();  // U block, z jumps and the stages are dead from here on
  unsigned char *zb[2] = {sm + L::SS, sm + L::U};
  if (tid == 0) {
    tma_store_wait_all();  // every Q slice of this CTA has reached global memory
#pragma unroll
    for (int k = 0; k < 2; ++k)
      if (k < N - 1) { mbar_expect_tx(&bar[4 + k], (uint32_t)L::Q_BYTES); tma_load_4d(zb[k], &tmQ, l0, 0, 3 * k, eb, &bar[4 + k]); }
  }
  double zq[2][3][NV];
#pragma unroll
  for (int s = 0; s < 2; ++s)
#pragma unroll
    for (int n = 0; n < 3; ++n)
#pragma unroll
      for (int a = 0; a < NV; ++a) zq[s][n][a] = 0.0;
#pragma unroll
  for (int k = 0; k < N; ++k) {
    const double *src = sQ;
    if (k < N - 1) {
      mbar_wait(&bar[4 + (k & 1)], (k >> 1) & 1);
      src = (const double *)zb[k & 1];
    }
#pragma unroll
    for (int n = 0; n < 3; ++n)
#pragma unroll
      for (int a = 0; a < NV; ++a) {
        const double q = src[((n * NFP + ij) * NV + a) * E + el];
        zq[0][n][a] = fma(op.lm[k], q, zq[0][n][a]);
        zq[1][n][a] = fma(op.lp[k], q, zq[1][n][a]);
      }
    if (k + 2 < N - 1) {  // refill this buffer with slice k + 2
      __syncthreads();
      if (tid == 0) { mbar_expect_tx(&bar[4 + (k & 1)], (uint32_t)L::Q_BYTES); tma_load_4d(zb[k & 1], &tmQ, l0, 0, 3 * (k + 2), eb, &bar[4 + (k & 1)]); }
    }
  }
#pragma unroll
  for (int s = 0; s < 2; ++s) {
    if (!need_z[s]) continue;
    const int fp = (4 + s) * NFP + ij;
    double nrm[3], G[NV];
#pragma unroll
    for (int n = 0; n < 3; ++n) nrm[n] = fp_n[fp_row(true, ld, 3 * NF, n * NF + fp, e)];
    const int pe = BND ? fp_pe[fp_row(true, ld, NF, fp, e)] : 0;
    if constexpr (BND) face_visc<BND>(ufz[s], zq[s], nrm, ph, pe, bcs, G);
    else visc_normal_stream(ufz[s], nrm, ph, [&](int a, double *g) {
#pragma unroll
      for (int n = 0; n < 3; ++n) g[n] = zq[s][n][a];
    }, G);
#pragma unroll
    for (int a = 0; a < NV; ++a) gf[fp_row(true, ld, NF * NV, fp * NV + a, e)] = G[a];
  }
}

// ---------------------------------------------------------------------------------------------
// host side: tensor maps and launches
// ---------------------------------------------------------------------------------------------
template <int N, int E>
struct Maps {
  CUtensorMap U, S, R1, J, Jz, Q;
};

template <int N, int E, typename T>
bool make_maps(const DevConsts &c, const void *u, const double *jump, Maps<N, E> &m, const double *q) {
  constexpr int NFP = N * N, NU = N * NFP;
  static_assert(FR_BLK % E == 0, "a CTA's elements must lie in one element block");
  const uint64_t ld = (uint64_t)c.ld;
  bool ok = encode3(&m.U, sizeof(T) == 8, u, ld, NFP * NV, N, ld, (uint64_t)NFP * NV * ld, E, NFP * NV, N);  // caller layout
  ok = ok && encode_blk(&m.S, c.smat, ld, NU, 9, E, NFP, 9, c.aff ? 1 : 0);
  ok = ok && encode_blk(&m.R1, c.rcpj, ld, NFP, N, E, NFP, 1, c.aff ? 2 : 0);
  ok = ok && encode_blk(&m.J, jump, ld, NFP * NV, 6, E, N * NV, 4);
  ok = ok && encode_blk(&m.Jz, jump, ld, NFP * NV, 6, E, NFP * NV, 2);
  if (q) ok = ok && encode_blk(&m.Q, q, ld, NV * NFP, 3 * N, E, NV * NFP, 3);
  else m.Q = m.R1;
  return ok;
}

template <int N, int E, bool BND, bool SQ, typename T, int MINB>
cudaError_t launch_gradface_k(const DevConsts &c, const Maps<N, E> &m, const Ops1D<N> &op, const double *jump, double *gf, cudaStream_t s) {
  using L = GfLay<N, E, T>;
  auto kern = k_hex_gradface<N, E, BND, SQ, T, MINB>;
  static DevFlags done;
  cudaError_t err = set_smem(kern, L::TOTAL, done, c.dev);
  if (err != cudaSuccess) return err;
  kern<<<(unsigned)((c.Nel + E - 1) / E), N * N * E, L::TOTAL, s>>>(m.U, m.S, m.R1, m.J, m.Q, m.Jz, op, c.ph, jump, c.fp_n, c.fp_pe, c.face_need, c.bcs, gf,
                                                                  c.ld,
                                                                  c.Nel);
  return cudaGetLastError();
}

template <int N, int E, typename T>
cudaError_t launch_gradface(const DevConsts &c, const double *h_ops, const void *u, const double *jump, double *gf, double *q,
                            cudaStream_t s) {
  using L = GfLay<N, E, T>;
  static_assert(L::TOTAL <= SMEM_MAX, "shared memory");
  constexpr int MINB = min_blocks(L::TOTAL, N * N * E);
  Maps<N, E> m;
  if (!make_maps<N, E, T>(c, u, jump, m, q)) return cudaErrorNotSupported;
  const Ops1D<N> op = make_ops<N>(h_ops);
  if (!q) return cudaErrorInvalidValue;  // the z-face pass re-reads the stored Q slices
  return c.nbnd ? launch_gradface_k<N, E, true, true, T, MINB>(c, m, op, jump, gf, s) : launch_gradface_k<N, E, false, true, T, MINB>(c, m, op, jump, gf, s);
}

template <int N, typename T>
constexpr bool fits() {
  return GfLay<N, Cfg<N>::E, T>::TOTAL <= SMEM_MAX && N * N * Cfg<N>::E <= 1024;
}

template <int N, typename T>
cudaError_t gradface_n(const DevConsts &c, const double *h_ops, const void *u, const double *jump, double *gf, double *q, cudaStream_t s) {
  if constexpr (fits<N, T>()) {
    return launch_gradface<N, Cfg<N>::E, T>(c, h_ops, u, jump, gf, q, s);
  } else {
    return cudaErrorNotSupported;
  }
}

}  // namespace

bool hex_tma_supported(int n, bool f64) {
  if (!encoder() || !hex_tma_fluxdiv_supported(n, f64)) return false;
  switch (n) {
#define FR_CASE(NN) case NN: return f64 ? fits<NN, double>() : fits<NN, float>();
    FR_CASE(2) FR_CASE(3) FR_CASE(4) FR_CASE(5) FR_CASE(6) FR_CASE(7)
#undef FR_CASE
    default: return false;
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
