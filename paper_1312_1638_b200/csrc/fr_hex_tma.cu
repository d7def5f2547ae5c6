// TMA-fed, mbarrier-pipelined "z-slab" kernel for hexahedral elements (sm_100a): parts (2)-(3) of the Navier-Stokes
// right-hand side and the viscous half of part (5) (BASELINE.json north_star) in ONE launch.
//
//   k_hex_gradface : common solution and its jump at the element's own flux points (Eq 7, 25), gathered from the partner's
//                    U^f;  Q = J^-T {M4 U + M6 (C - U^f)} at the solution points (Eq 9-10 / Eq 42 :753), stored slice-major for
//                    k_hex_fluxdiv_tma;  Q interpolated to the element's own flux points (Eq 11 / Eq 43 :764) and contracted at
//                    once with the outward unit normal: G^f = n . f_vis(U^f, Q^f)  (Eq 22-24, the viscous part of Eq 26-27).
//                    Q^f (3 N_V N_f) and the common solution C^f (N_V N_f) are never stored.  Boundary flux points get the
//                    complete LDG viscous flux with the ghost state of App C.
//   (k_hex_fluxdiv_tma, fr_hex_fluxdiv_tma.cu: F~ = S f(U, Q), R = -(1/J) {(M1 - M3 M2) F~ + M3 D~}.)
//
// The jump C - U^f of Eq 9 at a flux point is  w_f (u_partner - u_own)  with  w_f = 1/2 + beta on the L side of its interface
// and 1/2 - beta on the R side (Eq 25): it needs the partner's U^f only where w_f != 0 (the paper's beta = 1/2: on L sides), and
// the same faces are the ones whose G^f carries a non-zero LDG weight (Eq 27).  The partner values are gathered by per-thread
// cp.async copies issued one slice ahead (offsets from the element-centric table fp_poff); there is no separate
// common-solution kernel and no jump array in HBM.
//
// Arithmetic: in the context's storage precision T.  Everything this kernel produces (Q, G^f) enters the right-hand side
// through the viscous flux only, whose share of the RHS is O(1/Re_h): single-precision arithmetic on the perturbation
// variables (O(1) values) keeps the single-precision bar of 1e-5 with a wide margin, and avoids a float <-> double conversion
// per shared-memory operand.  The inviscid path (k_hex_interp_tma, the pair kernels, k_hex_fluxdiv_tma) computes in double.
//
// Data movement: a CTA owns E consecutive elements.  The U block of those elements ([N_u*N_V] rows of E values) is brought
// into shared memory by ONE 3-D TMA box load; the metric terms S (9 rows per point) and 1/J stream slice by slice (z = k)
// through TMA box loads completing on mbarriers, issued ahead by one thread, so HBM latency is covered without registers or
// occupancy.  Thread (e, i, j) owns the column of points (i, j, .); contractions along x and y read shared memory,
// contractions along z use operator entries from the constant bank.
#include "fr_tma.cuh"

namespace fr {
namespace {

// ---------------------------------------------------------------------------------------------
// shared-memory layout (byte offsets from a 128-byte aligned base)
// ---------------------------------------------------------------------------------------------
// NST: depth of the {1/J, x/y partner values} ring (2; 1 where the second stage would cost the second resident CTA: p = 6 in double)
template <int N, int E, typename T, int NST = 2>
struct GfLay {
  static constexpr int NFP = N * N, NU = N * NFP;
  static constexpr size_t BAR = 0;
  static constexpr size_t OPS = 128;  // sD [N*N], sL [2][N], sGm [N], sGp [N]
  static constexpr size_t U = OPS + al128((N * N + 4 * N) * 8);
  static constexpr uint32_t U_TX = NU * NV * E * sizeof(T);
  static constexpr size_t PZ = U + al128(U_TX);                   // partner U^f of the two z faces [2][NFP][NV][E], then their jumps
  static constexpr size_t PZ_BYTES = 2 * NFP * NV * E * sizeof(T);
  static constexpr size_t SS = PZ + al128(PZ_BYTES);              // S of the current slice: ONE buffer, refilled during the face phase
  static constexpr uint32_t S_TX = 9 * NFP * E * sizeof(T), R_TX = NFP * E * sizeof(T);  // metric terms in the storage precision
  static constexpr size_t ST = SS + al128(S_TX);                  // two stages of {1/J (TMA), partner U^f of the x/y faces -> jumps (cp.async)}
  static constexpr size_t ST_P = al128(R_TX);
  static constexpr size_t P_BYTES = 4 * N * NV * E * sizeof(T);   // [slot 0..3 = faces 1, 3, 0, 2][N][NV][E]
  static constexpr size_t ST_BYTES = ST_P + al128(P_BYTES);
  static constexpr size_t Q = ST + NST * ST_BYTES;
  static constexpr size_t Q_BYTES = 3 * NV * NFP * E * sizeof(T);
  static constexpr size_t TOTAL = Q + al128(Q_BYTES) + 128;
};

// ---------------------------------------------------------------------------------------------
// k_hex_gradface
// ---------------------------------------------------------------------------------------------
// tmU: u as (ld, NFP*NV, N) box (E, NFP*NV, N); tmS: smat blocked, box (E, NFP, 9); tmR: rcpj blocked, box (E, NFP, 1);
// tmQ: Q workspace as (lane, NV*NFP, 3N, block), box (E, NV*NFP, 3): slice k, component n, point ij, variable a.
// uf: U^f of all elements in perturbation variables (k_hex_interp_tma), element-blocked; fp_poff: for every flux point the
// offset of its partner's first variable in uf, or -1 - bc_id on a boundary; face_code [6][ld]: 0 = no LDG weight (skip),
// 1 = L side (1/2 + beta), 2 = R side (1/2 - beta), 3 = boundary.
// AFF: affine mesh (one set of metric terms per element): S and 1/J are read once per thread from the per-element tables
// ([block][9][FR_BLK], [block][1][FR_BLK], fr_api.cu) instead of streaming through the ring.
template <int N, int E, bool BND, typename T, int MINB, int NST, bool AFF>
__global__ void __launch_bounds__(N *N *E, MINB)
    k_hex_gradface(const __grid_constant__ CUtensorMap tmU, const __grid_constant__ CUtensorMap tmS,
                   const __grid_constant__ CUtensorMap tmR, const __grid_constant__ CUtensorMap tmQ, Ops1D<N, T> op, Phys ph,
                   const T *__restrict__ uf, const int64_t *__restrict__ fp_poff, const T *__restrict__ fp_n,
                   const uint8_t *__restrict__ face_code, const BcDev *__restrict__ bcs, T *__restrict__ gf, const T *__restrict__ smat,
                   const T *__restrict__ rcpj, int64_t ld, int64_t Nel) {
  using L = GfLay<N, E, T, NST>;
  using R = T;  // arithmetic type of this kernel: the gradient feeds the viscous flux only (see the header comment)
  constexpr int NFP = N * N, NF = 6 * NFP;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  unsigned char *sm = smem_raw + ((128u - (smem_addr(smem_raw) & 127u)) & 127u);  // stays in the shared address space
  uint64_t *bar = (uint64_t *)(sm + L::BAR);
  R *sD = (R *)(sm + L::OPS), *sL = sD + N * N;  // sL[0][m] = l_m(-1), sL[1][m] = l_m(+1)
  R *sGm = sL + 2 * N, *sGp = sGm + N;
  T *sU = (T *)(sm + L::U);
  T *sPz = (T *)(sm + L::PZ);
  const T *stS = (const T *)(sm + L::SS);
  unsigned char *sSt = sm + L::ST;
  T *sQ = (T *)(sm + L::Q);  // [3][NFP][NV][E]
  const int tid = threadIdx.x, el = tid % E, ij = patch_ij<N>(tid / E), i = ij % N, j = ij / N;  // 2 x 2 patches per warp (fr_tma.cuh)
  const int e0 = blockIdx.x * E, l0 = e0 % FR_BLK, eb = e0 / FR_BLK;  // first element: lane and element block (fp_row)
  const int64_t e = (int64_t)e0 + el;
  const bool act = e < Nel;
  const R wL = (R)(0.5 + ph.beta), wR = (R)(0.5 - ph.beta);

  if (tid == 0) {
    mbar_init(&bar[0], 1); mbar_init(&bar[1], 1); mbar_init(&bar[2], 1); mbar_init(&bar[3], 1);
    mbar_init(&bar[4], 1); mbar_init(&bar[5], 1);  // second pass over the Q slices (z faces)
    fence_barrier_init();
    fence_proxy_async();
  }
  for (int t = tid; t < N * N; t += NFP * E) sD[t] = op.D[t];
  for (int t = tid; t < N; t += NFP * E) { sL[t] = op.lm[t]; sL[N + t] = op.lp[t]; sGm[t] = op.gm[t]; sGp[t] = op.gp[t]; }
  __syncthreads();
  auto issue_R = [&](int s, int k) {
    mbar_expect_tx(&bar[1 + s], L::R_TX);
    tma_load_4d(sSt + s * L::ST_BYTES, &tmR, l0, 0, k, eb, &bar[1 + s]);
  };
  auto issue_S = [&](int k) {
    mbar_expect_tx(&bar[3], L::S_TX);
    tma_load_4d(sm + L::SS, &tmS, l0, NFP * k, 0, eb, &bar[3]);
  };
  if (tid == 0) {
    mbar_expect_tx(&bar[0], L::U_TX);
    tma_load_3d(sm + L::U, &tmU, e0, 0, 0, &bar[0]);
    if (!AFF) {
      issue_S(0);
      issue_R(0, 0);
      if (NST > 1 && N > 1) issue_R(1, 1);
    }
  }
  // x/y-face tasks of a thread per slice: task t = ij + q NFP < 4 N handles flux point (slot t / N, line m = t % N) of the
  // thread's element; slots 0..3 = faces 1, 3 (+x, +y: the L sides of structured meshes, so that skipped tasks fall into the
  // same warps), then 0, 2.  code: 0 skip, 1 / 2 interior with weight 1/2 +- beta, 3 boundary.
  constexpr int TPT = (4 * N + NFP - 1) / NFP;
  auto face_of = [](int t) { return t < 2 * N ? 2 * (t / N) + 1 : 2 * (t / N - 2); };
  int code_xy[TPT];
  int64_t off_nx[TPT];  // partner offset of the task's flux point in the next slice to gather
#pragma unroll
  for (int q = 0; q < TPT; ++q) {
    const int t = ij + q * NFP;
    code_xy[q] = (t < 4 * N && act) ? face_code[(size_t)face_of(t) * ld + e] : 0;
    off_nx[q] = 0;
  }
  int code_z[2];
#pragma unroll
  for (int s = 0; s < 2; ++s) code_z[s] = act ? face_code[(size_t)(4 + s) * ld + e] : 0;

  // element-blocked tables (fp_row): all elements of a CTA lie in one element block, so a row of the CTA's elements starts at
  // (block base, CTA-uniform 64-bit) + row * FR_BLK + lane (32-bit per-thread index)
  const int lane = l0 + el;
  const int64_t *poff_blk = fp_poff + (size_t)eb * NF * FR_BLK;
  const T *fpn_blk = fp_n + (size_t)eb * (3 * NF) * FR_BLK;
  T *gf_blk = gf + (size_t)eb * (NF * NV) * FR_BLK;
  auto poff = [&](int fp) { return poff_blk[fp * FR_BLK + lane]; };
  // gather of the partner's U^f (N_V values) of one flux point: per-thread asynchronous copies, consumed by the same thread
  auto gather = [&](T *dst, int64_t off) {
#pragma unroll
    for (int a = 0; a < NV; ++a) cp_async<sizeof(T)>(dst + a * E, uf + off + (int64_t)a * FR_BLK);
  };
  auto gather_xy = [&](int k, int64_t *off) {  // slice k into stage k % NST
    T *sP = (T *)(sSt + (k % NST) * L::ST_BYTES + L::ST_P);
#pragma unroll
    for (int q = 0; q < TPT; ++q) {
      const int t = ij + q * NFP;
      if (code_xy[q] == 1 || code_xy[q] == 2) gather(sP + (size_t)t * NV * E + el, off[q]);
    }
  };
  {
    // Every table entry the prologue needs is loaded first, independent of the face codes (the table holds an offset for every
    // flux point), so that the codes and the offsets of the z faces and of slices 0 .. NST come back in ONE round trip instead
    // of four dependent ones (the cp.async statements below are ordering points for the compiler).
    int64_t offz[2], offk[NST][TPT];
#pragma unroll
    for (int s = 0; s < 2; ++s) offz[s] = poff((4 + s) * NFP + ij);
#pragma unroll
    for (int k1 = 0; k1 < NST; ++k1)
#pragma unroll
      for (int q = 0; q < TPT; ++q) {
        const int t = ij + q * NFP;
        offk[k1][q] = (t < 4 * N && k1 < N) ? poff(face_of(t) * NFP + t % N + N * k1) : 0;
      }
    if (N > NST) {
#pragma unroll
      for (int q = 0; q < TPT; ++q) {
        const int t = ij + q * NFP;
        off_nx[q] = t < 4 * N ? poff(face_of(t) * NFP + t % N + N * NST) : 0;
      }
    }
    // z faces and slice 0 (group 0), slices 1 .. NST - 1 (one group each); the offsets of slice NST wait in registers
#pragma unroll
    for (int s = 0; s < 2; ++s)
      if (code_z[s] == 1 || code_z[s] == 2) gather(sPz + (size_t)(s * NFP + ij) * NV * E + el, offz[s]);
    gather_xy(0, offk[0]);
    cp_async_commit();
#pragma unroll
    for (int k1 = 1; k1 < NST; ++k1) {
      if (k1 < N) gather_xy(k1, offk[k1]);
      cp_async_commit();
    }
  }
  // jump C - U^f (Eq 9) from the partner's U^f and the own interpolated state, both in the perturbation variables w (whose
  // gradient this kernel takes); boundary: C = (1/2 - beta) u + (1/2 + beta) B_ldg u  (:797)
  auto jump_of = [&](int code, int64_t off_or_bc, const R *uown, T *slot) {
    R d[NV];
    if (code == 1 || code == 2) {
      const R w = code == 1 ? wL : wR;
#pragma unroll
      for (int a = 0; a < NV; ++a) d[a] = w * ((R)slot[a * E] - uown[a]);
    } else if (BND && code == 3) {
      double uw[NV], uc[NV], gi[NV], gl[NV];
#pragma unroll
      for (int a = 0; a < NV; ++a) uw[a] = (double)uown[a];
      from_pert<3>(ph, uw, uc);
      ghost_states<3>(bcs[-1 - off_or_bc], uc, ph.gamma, gi, gl);
      to_pert<3>(ph, gl, gl);
#pragma unroll
      for (int a = 0; a < NV; ++a) d[a] = wL * ((R)gl[a] - uown[a]);
    } else {
#pragma unroll
      for (int a = 0; a < NV; ++a) d[a] = 0;
    }
#pragma unroll
    for (int a = 0; a < NV; ++a) slot[a * E] = (T)d[a];
  };
  // own state at the x/y flux point of task t in slice k (interpolation along its line, Eq 6)
  auto own_xy = [&](int t, int k, R *uo) {
    const int slot = t / N, m = t % N;
    const int base = NFP * k + (slot % 2 == 0 ? m * N : m), stride = slot % 2 == 0 ? 1 : N;  // slots 0, 2: x faces (line j = m)
    const R *lc = sL + (slot < 2 ? N : 0);
#pragma unroll
    for (int a = 0; a < NV; ++a) uo[a] = 0;
#pragma unroll
    for (int mm = 0; mm < N; ++mm) {
      const R l = lc[mm];
#pragma unroll
      for (int a = 0; a < NV; ++a) uo[a] = fma(l, (R)sU[((size_t)(base + mm * stride) * NV + a) * E + el], uo[a]);
    }
  };
  // own state at the task's flux point, kept from phase A (jump) to phase C (G^f) of the same slice when a thread has one task
  constexpr bool KEEP = TPT == 1;
  R uo_keep[KEEP ? NV : 1];
  auto phase_A = [&](int k) {  // jumps of the x/y faces of slice k, in place over the gathered partner values
    T *sP = (T *)(sSt + (k % NST) * L::ST_BYTES + L::ST_P);
#pragma unroll
    for (int q = 0; q < TPT; ++q) {
      const int t = ij + q * NFP;
      if (t >= 4 * N) continue;
      R uo[NV];
      if (code_xy[q] != 0) own_xy(t, k, uo);
      if constexpr (KEEP) {
#pragma unroll
        for (int a = 0; a < NV; ++a) uo_keep[a] = uo[a];
      }
      int64_t bc = 0;
      if (BND && code_xy[q] == 3) bc = poff(face_of(t) * NFP + t % N + N * k);
      jump_of(code_xy[q], bc, uo, sP + (size_t)t * NV * E + el);
    }
  };
  R S_el[3][3], rj_el = 0;
  if (AFF) {
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
      for (int b = 0; b < 3; ++b) S_el[a][b] = (R)smat[((size_t)eb * 9 + a * 3 + b) * FR_BLK + lane];
    rj_el = (R)rcpj[(size_t)eb * FR_BLK + lane];
  }
  mbar_wait(&bar[0], 0);
  if (ph.rho0 != 0.0) {
    // the U block becomes w = T (u - u_ref) in place (fr_physics.cuh): every thread converts its own column
#pragma unroll
    for (int m = 0; m < N; ++m) {
      double w[NV];
      T *col = sU + ((size_t)(NFP * m + ij) * NV) * E + el;
#pragma unroll
      for (int a = 0; a < NV; ++a) w[a] = (double)col[a * E];
      if (act) to_pert<3>(ph, w, w);
#pragma unroll
      for (int a = 0; a < NV; ++a) col[a * E] = (T)w[a];
    }
    __syncthreads();
  }
  // the thread's own column (i, j, .) of w for the contractions along z: in registers in single precision (25 registers; 1.6 %
  // off the kernel on C3), read from the U block in double precision (50 registers more than the 128 that two resident CTAs
  // of 7 warps allow: 0.35 -> 0.42 ms with the spills)
  constexpr bool ZREG = sizeof(T) == 4 && !BND && N <= 6;  // (the boundary instantiations and p = 6 would spill)
  R wcol[ZREG ? N : 1][NV];
  if constexpr (ZREG) {
#pragma unroll
    for (int m = 0; m < N; ++m)
#pragma unroll
      for (int a = 0; a < NV; ++a) wcol[m][a] = (R)sU[((size_t)(NFP * m + ij) * NV + a) * E + el];
  }
  auto wz = [&](int m, int a) -> R {
    if constexpr (ZREG) return wcol[m][a];
    else return (R)sU[((size_t)(NFP * m + ij) * NV + a) * E + el];
  };
  cp_async_wait<NST - 1>();  // z faces and slice 0 have arrived (this thread's own copies)
  {
    R uz[2][NV];
#pragma unroll
    for (int s = 0; s < 2; ++s)
#pragma unroll
      for (int a = 0; a < NV; ++a) uz[s][a] = 0;
#pragma unroll
    for (int m = 0; m < N; ++m)
#pragma unroll
      for (int a = 0; a < NV; ++a) {
        const R v = wz(m, a);
        uz[0][a] = fma(op.lm[m], v, uz[0][a]);
        uz[1][a] = fma(op.lp[m], v, uz[1][a]);
      }
#pragma unroll
    for (int s = 0; s < 2; ++s) {
      int64_t bc = 0;
      if (BND && code_z[s] == 3) bc = poff((4 + s) * NFP + ij);
      jump_of(code_z[s], bc, uz[s], sPz + (size_t)(s * NFP + ij) * NV * E + el);
    }
  }
  phase_A(0);
  __syncthreads();  // jumps of the z faces and of slice 0 are visible

#pragma unroll
  for (int k = 0; k < N; ++k) {
    // own outward normals of the slice's x/y flux points (global, element-blocked): requested here, consumed in the face phase
    T nrm_pf[TPT][3];
#pragma unroll
    for (int q = 0; q < TPT; ++q) {
      const int t = ij + q * NFP;
#pragma unroll
      for (int n = 0; n < 3; ++n)
        nrm_pf[q][n] = code_xy[q] != 0 ? fpn_blk[(n * NF + face_of(t) * NFP + t % N + N * k) * FR_BLK + lane] : (T)0;
    }
    if (!AFF) {
      mbar_wait(&bar[1 + (k % NST)], (k / NST) & 1);
      mbar_wait(&bar[3], k & 1);
    }
    const T *stR = (const T *)(sSt + (k % NST) * L::ST_BYTES);
    const T *stJ = (const T *)(sSt + (k % NST) * L::ST_BYTES + L::ST_P);  // [slot][line][NV][E]: slots 0, 1 = +x, +y; 2, 3 = -x, -y
    const T *su = sU + (size_t)(NFP * k) * NV * E + el;  // slice k
    {
      R S[3][3];
#pragma unroll
      for (int a = 0; a < 3; ++a)
#pragma unroll
        for (int b = 0; b < 3; ++b) S[a][b] = AFF ? S_el[a][b] : (R)stS[((a * 3 + b) * NFP + ij) * E + el];
      const R rj = AFF ? rj_el : (R)stR[ij * E + el];
      const R gmi = sGm[i], gpi = sGp[i], gmj = sGm[j], gpj = sGp[j];
#pragma unroll
      for (int a = 0; a < NV; ++a) {
        // M6 = n~ (x) M3 (A1): the reference normal is -1 on the -1 faces (jumps of faces without an LDG weight are zero;
        // skipping their reads under a predicate was 4 % slower)
        R qx = fma(gpi, (R)stJ[((0 * N + j) * NV + a) * E + el], -gmi * (R)stJ[((2 * N + j) * NV + a) * E + el]);
        R qy = fma(gpj, (R)stJ[((1 * N + i) * NV + a) * E + el], -gmj * (R)stJ[((3 * N + i) * NV + a) * E + el]);
        R qz = fma(op.gp[k], (R)sPz[((1 * NFP + ij) * NV + a) * E + el], -op.gm[k] * (R)sPz[((0 * NFP + ij) * NV + a) * E + el]);
#pragma unroll
        for (int m = 0; m < N; ++m) {
          qx = fma(sD[i * N + m], (R)su[((j * N + m) * NV + a) * E], qx);
          qy = fma(sD[j * N + m], (R)su[((m * N + i) * NV + a) * E], qy);
          qz = fma(op.D[k * N + m], wz(m, a), qz);
        }
        R q3[3];
        to_physical(S, rj, qx, qy, qz, q3);
#pragma unroll
        for (int n = 0; n < 3; ++n) sQ[((n * NFP + ij) * NV + a) * E + el] = (T)q3[n];
      }
    }
    fence_proxy_async();  // make the sQ writes visible to the bulk store
    __syncthreads();      // Q of the slice is complete; S, 1/J and the jumps of stage k&1 have been consumed
    if (!AFF && tid == 0 && k + 1 < N) issue_S(k + 1);
    if (!AFF && tid == 0 && k + NST < N) issue_R(k % NST, k + NST);
    if (tid == 0) { tma_store_4d(&tmQ, l0, 0, 3 * k, eb, sQ); tma_store_commit(); }
    if (k + NST < N) {  // partner values of slice k + NST into the freed stage; the offsets of the slice after it start their way
      gather_xy(k + NST, off_nx);
      if (k + NST + 1 < N) {
#pragma unroll
        for (int q = 0; q < TPT; ++q) {
          const int t = ij + q * NFP;
          off_nx[q] = (code_xy[q] == 1 || code_xy[q] == 2) ? poff(face_of(t) * NFP + t % N + N * (k + NST + 1)) : 0;
        }
      }
    }
    cp_async_commit();
    // x / y faces of the slice: G^f at the flux points that carry an LDG weight, one thread each
#pragma unroll
    for (int q = 0; q < TPT; ++q) {
      if (code_xy[q] == 0) continue;
      const int t = ij + q * NFP;
      const int slot = t / N, f = face_of(t), m = t % N;
      const int base = slot % 2 == 0 ? m * N : m, stride = slot % 2 == 0 ? 1 : N;
      const R *lc = sL + (slot < 2 ? N : 0);
      const int fp = f * NFP + m + N * k;
      R nrm[3], uo[NV], G[NV];
#pragma unroll
      for (int n = 0; n < 3; ++n) nrm[n] = (R)nrm_pf[q][n];
      if constexpr (KEEP) {
#pragma unroll
        for (int a = 0; a < NV; ++a) uo[a] = uo_keep[a];
      } else {
        own_xy(t, k, uo);
      }
      if constexpr (BND) {
        const int pe = code_xy[q] == 3 ? (int)poff(fp) : 0;
        R qf[3][NV];
#pragma unroll
        for (int n = 0; n < 3; ++n)
#pragma unroll
          for (int a = 0; a < NV; ++a) {
            R qq = 0;
#pragma unroll
            for (int mm = 0; mm < N; ++mm) qq = fma(lc[mm], (R)sQ[((n * NFP + base + mm * stride) * NV + a) * E + el], qq);
            qf[n][a] = qq;
          }
        face_visc_r<BND, R>(uo, qf, nrm, ph, pe, bcs, G);
      } else {
        visc_normal_stream<R>(uo, nrm, ph, [&](int a, R *g) {
#pragma unroll
          for (int n = 0; n < 3; ++n) {
            R qq = 0;
#pragma unroll
            for (int mm = 0; mm < N; ++mm) qq = fma(lc[mm], (R)sQ[((n * NFP + base + mm * stride) * NV + a) * E + el], qq);
            g[n] = qq;
          }
        }, G);
      }
#pragma unroll
      for (int a = 0; a < NV; ++a) gf_blk[(fp * NV + a) * FR_BLK + lane] = (T)G[a];
    }
    if (k + 1 < N) {
      cp_async_wait<NST - 1>();  // slice k + 1 has arrived (with two stages slice k + 2 may still be in flight)
      phase_A(k + 1);
    }
    if (tid == 0) tma_store_wait_read();  // the bulk store has read sQ
    if (k + 1 < N) __syncthreads();  // jumps of slice k + 1 visible; sQ free
  }
  // ---- z faces.  Q^f on them is sum_k l(+-1)_k Q(i, j, k): instead of carrying 2 x 15 accumulators through the slice
  // loop, the Q slices just stored are streamed once more (TMA loads, L2 hits) through two buffers that the slice loop
  // no longer needs: [SS .. Q) (S, 1/J, x/y jumps) and [U .. SS) (U block, z jumps).  The last slice is still in sQ.
  constexpr bool ZB_IN_U = L::SS - L::U >= 2 * al128(L::Q_BYTES);  // both reload buffers inside the U block + z jumps
  static_assert(ZB_IN_U || (L::Q - L::SS >= L::Q_BYTES && L::SS - L::U >= L::Q_BYTES), "Q slice does not fit the reused buffers");
  R ufz[2][NV];
#pragma unroll
  for (int s = 0; s < 2; ++s)
#pragma unroll
    for (int a = 0; a < NV; ++a) ufz[s][a] = 0;
#pragma unroll
  for (int m = 0; m < N; ++m)
#pragma unroll
    for (int a = 0; a < NV; ++a) {
      const R v = wz(m, a);
      ufz[0][a] = fma(op.lm[m], v, ufz[0][a]);
      ufz[1][a] = fma(op.lp[m], v, ufz[1][a]);
    }
  // The reload buffers are written by the async proxy (TMA) after they were read through the generic proxy: the proxy fence
  // before each barrier orders those reads before the bulk copy that the barrier releases.  Without it a shared-memory load
  // issued before the barrier, whose value only feeds register accumulators, may still be in flight when the copy lands
  // (seen in single precision: G^f of a z face differed from run to run in a few warps per launch).
  fence_proxy_async();
  __syncthreads();  // U block, z jumps and the stages are dead from here on
  unsigned char *zb[2] = {ZB_IN_U ? sm + L::U : sm + L::SS, ZB_IN_U ? sm + L::U + al128(L::Q_BYTES) : sm + L::U};
  if (tid == 0) {
    tma_store_wait_all();  // every Q slice of this CTA has reached global memory
#pragma unroll
    for (int k = 0; k < 2; ++k)
      if (k < N - 1) { mbar_expect_tx(&bar[4 + k], (uint32_t)L::Q_BYTES); tma_load_4d(zb[k], &tmQ, l0, 0, 3 * k, eb, &bar[4 + k]); }
  }
  T nrm_z[2][3];  // own normals of the z flux points: requested before the reload loop
  int pe_z[2];
#pragma unroll
  for (int s = 0; s < 2; ++s) {
#pragma unroll
    for (int n = 0; n < 3; ++n) nrm_z[s][n] = code_z[s] != 0 ? fpn_blk[(n * NF + (4 + s) * NFP + ij) * FR_BLK + lane] : (T)0;
    pe_z[s] = (BND && code_z[s] == 3) ? (int)poff((4 + s) * NFP + ij) : 0;
  }
  R zq[2][3][NV];
#pragma unroll
  for (int s = 0; s < 2; ++s)
#pragma unroll
    for (int n = 0; n < 3; ++n)
#pragma unroll
      for (int a = 0; a < NV; ++a) zq[s][n][a] = 0;
#pragma unroll
  for (int k = 0; k < N; ++k) {
    const T *src = sQ;
    if (k < N - 1) {
      mbar_wait(&bar[4 + (k & 1)], (k >> 1) & 1);
      src = (const T *)zb[k & 1];
    }
#pragma unroll
    for (int n = 0; n < 3; ++n)
#pragma unroll
      for (int a = 0; a < NV; ++a) {
        const R q = (R)src[((n * NFP + ij) * NV + a) * E + el];
        zq[0][n][a] = fma(op.lm[k], q, zq[0][n][a]);
        zq[1][n][a] = fma(op.lp[k], q, zq[1][n][a]);
      }
    if (k + 2 < N - 1) {  // refill this buffer with slice k + 2
      fence_proxy_async();  // this thread's reads of the buffer are ordered before the refill (see above)
      __syncthreads();
      if (tid == 0) { mbar_expect_tx(&bar[4 + (k & 1)], (uint32_t)L::Q_BYTES); tma_load_4d(zb[k & 1], &tmQ, l0, 0, 3 * (k + 2), eb, &bar[4 + (k & 1)]); }
    }
  }
#pragma unroll
  for (int s = 0; s < 2; ++s) {
    if (code_z[s] == 0) continue;
    const int fp = (4 + s) * NFP + ij;
    R nrm[3], G[NV];
#pragma unroll
    for (int n = 0; n < 3; ++n) nrm[n] = (R)nrm_z[s][n];
    const int pe = pe_z[s];
    if constexpr (BND) face_visc_r<BND, R>(ufz[s], zq[s], nrm, ph, pe, bcs, G);
    else visc_normal_stream<R>(ufz[s], nrm, ph, [&](int a, R *g) {
#pragma unroll
      for (int n = 0; n < 3; ++n) g[n] = zq[s][n][a];
    }, G);
#pragma unroll
    for (int a = 0; a < NV; ++a) gf_blk[(fp * NV + a) * FR_BLK + lane] = (T)G[a];
  }
}

// ---------------------------------------------------------------------------------------------
// host side: tensor maps and launches
// ---------------------------------------------------------------------------------------------
struct Maps {
  CUtensorMap U, S, R1, Q;
};

template <int N, int E, typename T>
bool make_maps(const DevConsts &c, const void *u, Maps &m, const void *q) {
  constexpr int NFP = N * N, NU = N * NFP;
  static_assert(FR_BLK % E == 0, "a CTA's elements must lie in one element block");
  const uint64_t ld = (uint64_t)c.ld;
  bool ok = encode3(&m.U, sizeof(T) == 8, u, ld, NFP * NV, N, ld, (uint64_t)NFP * NV * ld, E, NFP * NV, N);  // caller layout
  ok = ok && encode_blk(&m.S, sizeof(T) == 8, c.smat, ld, NU, 9, E, NFP, 9, c.aff ? 1 : 0);  // metric terms in T on this path (fr_api.cu)
  ok = ok && encode_blk(&m.R1, sizeof(T) == 8, c.rcpj, ld, NFP, N, E, NFP, 1, c.aff ? 2 : 0);
  ok = ok && encode_blk(&m.Q, sizeof(T) == 8, q, ld, NV * NFP, 3 * N, E, NV * NFP, 3);
  return ok;
}

template <int N, int E, bool BND, typename T, int MINB, int NST, bool AFF>
cudaError_t launch_gradface_k(const DevConsts &c, const Maps &m, const Ops1D<N, T> &op, const T *uf, T *gf, cudaStream_t s) {
  using L = GfLay<N, E, T, NST>;
  auto kern = k_hex_gradface<N, E, BND, T, MINB, NST, AFF>;
  static DevFlags done;
  cudaError_t err = set_smem(kern, L::TOTAL, done, c.dev);
  if (err != cudaSuccess) return err;
  kern<<<(unsigned)((c.Nel + E - 1) / E), N * N * E, L::TOTAL, s>>>(m.U, m.S, m.R1, m.Q, op, c.ph, uf, c.fp_poff, (const T *)c.fp_n, c.face_code, c.bcs, gf,
                                                                  (const T *)c.smat, (const T *)c.rcpj, c.ld, c.Nel);
  return cudaGetLastError();
}

template <int N, int E, typename T>
cudaError_t launch_gradface(const DevConsts &c, const double *h_ops, const void *u, const void *uf, void *gf, void *q, cudaStream_t s) {
  // one ring stage instead of two where that is what lets a second CTA reside on the SM (p = 6 in double precision: 121.6 -> 115.5 KB)
  constexpr int REGS = sizeof(T) == 8 ? 128 : 96;
  constexpr int NST = (min_blocks(GfLay<N, E, T, 2>::TOTAL, N * N * E, REGS) < 2 && min_blocks(GfLay<N, E, T, 1>::TOTAL, N * N * E, REGS) >= 2) ? 1 : 2;
  using L = GfLay<N, E, T, NST>;
  static_assert(L::TOTAL <= SMEM_MAX, "shared memory");
  constexpr int MINB = min_blocks(L::TOTAL, N * N * E, REGS);  // single-precision arithmetic needs fewer registers
  if (!q) return cudaErrorInvalidValue;  // the z-face pass re-reads the stored Q slices
  bool fresh = true;
  MapCache::Ent *ent = ((MapCache *)c.map_cache)->get(1, u, q, nullptr, fresh);
  Maps &m = *reinterpret_cast<Maps *>(ent->m);
  static_assert(sizeof(Maps) <= sizeof(ent->m), "map cache entry");
  if (fresh && !make_maps<N, E, T>(c, u, m, q)) { ent->id = -1; return cudaErrorNotSupported; }
  const Ops1D<N, T> op = make_ops<N, T>(h_ops);
  // the affine specialisation where it was measured to win (C5-shaped meshes: p = 6 3.07 -> 2.39 ms, p = 5 -4.9 %, p = 3, 4 -1 % in
  // double; p = 6 -4.5 % in single precision; p = 2 in double and p = 4, 5 in single precision lose 1 - 8 % with it)
  constexpr bool AFF_WINS = sizeof(T) == 8 ? N >= 4 : N == 7;
  if constexpr (AFF_WINS) {
    if (c.aff)
      return c.nbnd ? launch_gradface_k<N, E, true, T, MINB, NST, true>(c, m, op, (const T *)uf, (T *)gf, s)
                    : launch_gradface_k<N, E, false, T, MINB, NST, true>(c, m, op, (const T *)uf, (T *)gf, s);
  }
  return c.nbnd ? launch_gradface_k<N, E, true, T, MINB, NST, false>(c, m, op, (const T *)uf, (T *)gf, s)
                : launch_gradface_k<N, E, false, T, MINB, NST, false>(c, m, op, (const T *)uf, (T *)gf, s);
}

template <int N, typename T>
constexpr bool fits() {
  return GfLay<N, Cfg<N, T>::E_SLAB, T>::TOTAL <= SMEM_MAX && N * N * Cfg<N, T>::E_SLAB <= 1024;
}

template <int N, typename T>
cudaError_t gradface_n(const DevConsts &c, const double *h_ops, const void *u, const void *uf, void *gf, void *q, cudaStream_t s) {
  if constexpr (fits<N, T>()) {
    return launch_gradface<N, Cfg<N, T>::E_SLAB, T>(c, h_ops, u, uf, gf, q, s);
  } else {
    return cudaErrorNotSupported;
  }
}

}  // namespace

void *hex_tma_cache_create() { return new MapCache(); }
void hex_tma_cache_destroy(void *cache) { delete (MapCache *)cache; }

bool hex_tma_supported(int n, bool f64) {
  if (!encoder() || !hex_tma_fluxdiv_supported(n, f64)) return false;
  switch (n) {
#define FR_CASE(NN) case NN: return f64 ? fits<NN, double>() : fits<NN, float>();
    FR_CASE(2) FR_CASE(3) FR_CASE(4) FR_CASE(5) FR_CASE(6) FR_CASE(7)
#undef FR_CASE
    default: return false;
  }
}

cudaError_t hex_tma_gradface(const DevConsts &c, const double *h_ops, const void *u, const void *uf, void *gf, void *q, cudaStream_t s) {
  switch (c.n) {
#define FR_CASE(NN) case NN: return c.f64 ? gradface_n<NN, double>(c, h_ops, u, uf, gf, q, s) : gradface_n<NN, float>(c, h_ops, u, uf, gf, q, s);
    FR_CASE(2) FR_CASE(3) FR_CASE(4) FR_CASE(5) FR_CASE(6) FR_CASE(7)
#undef FR_CASE
    default: return cudaErrorNotSupported;
  }
}

}  // namespace fr
