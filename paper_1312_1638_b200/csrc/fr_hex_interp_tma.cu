// k_hex_interp_tma: U^f = M0 U on hexahedra (Eq 6 :186 / Eq 41 :745), part (1) of the right-hand side, as a TMA-fed
// (stored in the perturbation variables w = T (u - u_ref) of fr_physics.cuh; with no reference state w = u)
// z-slab kernel.  A CTA owns E consecutive elements; their whole U block ([N_u*N_V] rows of E values, caller layout)
// arrives by ONE 3-D TMA box load; thread (e, i, j) interpolates its column to the two z faces from shared memory,
// and the 4 N x/y-face flux points of every slice are interpolated along their lines by one thread each.  U^f is
// written element-blocked (fr_dev.hpp: fp_row) in the storage precision T of the context (all arithmetic in double).  Several CTAs are resident per SM (40 KB at p = 4), so the load of
// one CTA overlaps the arithmetic and the stores of the others.
#include "fr_tma.cuh"

namespace fr {
namespace {

template <int N, int E, typename T>
__global__ void __launch_bounds__(N *N *E) k_hex_interp_tma(const __grid_constant__ CUtensorMap tmU, Ops1D<N> op, Phys ph,
                                                            T *__restrict__ uf, int64_t ld, int64_t Nel) {
  constexpr int NFP = N * N, NU = N * NFP, NF = 6 * NFP;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  unsigned char *sm = smem_raw + ((128u - (smem_addr(smem_raw) & 127u)) & 127u);
  uint64_t *bar = (uint64_t *)sm;
  double *sL = (double *)(sm + 64);          // sL[0][m] = l_m(-1), sL[1][m] = l_m(+1)
  const T *sU = (const T *)(sm + 128 + al128(2 * N * 8));  // [NU*NV][E]
  const int tid = threadIdx.x, el = tid % E, ij = tid / E;
  const int e0 = blockIdx.x * E;
  const int64_t e = (int64_t)e0 + el;
  if (tid == 0) {
    mbar_init(bar, 1);
    fence_barrier_init();
    fence_proxy_async();
  }
  for (int t = tid; t < N; t += NFP * E) { sL[t] = op.lm[t]; sL[N + t] = op.lp[t]; }
  __syncthreads();
  if (tid == 0) {
    mbar_expect_tx(bar, NU * NV * E * sizeof(T));
    tma_load_3d(const_cast<T *>(sU), &tmU, e0, 0, 0, bar);
  }
  mbar_wait(bar, 0);
  if (e >= Nel) return;
  // z faces (4, 5): flux point ij, line = the column of the thread
  {
    double zm[NV], zp[NV];
#pragma unroll
    for (int a = 0; a < NV; ++a) zm[a] = zp[a] = 0.0;
#pragma unroll
    for (int m = 0; m < N; ++m) {
      double w[NV];
#pragma unroll
      for (int a = 0; a < NV; ++a) w[a] = (double)sU[((size_t)(NFP * m + ij) * NV + a) * E + el];
      to_pert<3>(ph, w, w);  // perturbation variables before the interpolation (fr_physics.cuh)
#pragma unroll
      for (int a = 0; a < NV; ++a) {
        zm[a] = fma(op.lm[m], w[a], zm[a]);
        zp[a] = fma(op.lp[m], w[a], zp[a]);
      }
    }
#pragma unroll
    for (int a = 0; a < NV; ++a) {
      uf[fp_row(true, ld, NF * NV, (4 * NFP + ij) * NV + a, e)] = (T)zm[a];
      uf[fp_row(true, ld, NF * NV, (5 * NFP + ij) * NV + a, e)] = (T)zp[a];
    }
  }
  // x / y faces: 4 N flux points per slice, N slices; task t = (slice k, face f, line m)
  for (int t = ij; t < 4 * N * N; t += NFP) {
    const int k = t / (4 * N), f = (t / N) % 4, m = t % N;
    const int base = NFP * k + (f < 2 ? m * N : m), stride = f < 2 ? 1 : N;
    const double *lc = sL + (f & 1) * N;
    double v[NV];
#pragma unroll
    for (int a = 0; a < NV; ++a) v[a] = 0.0;
#pragma unroll
    for (int mm = 0; mm < N; ++mm) {
      const double l = lc[mm];
      double w[NV];
#pragma unroll
      for (int a = 0; a < NV; ++a) w[a] = (double)sU[((size_t)(base + mm * stride) * NV + a) * E + el];
      to_pert<3>(ph, w, w);
#pragma unroll
      for (int a = 0; a < NV; ++a) v[a] = fma(l, w[a], v[a]);
    }
    const int fp = f * NFP + m + N * k;
#pragma unroll
    for (int a = 0; a < NV; ++a) uf[fp_row(true, ld, NF * NV, fp * NV + a, e)] = (T)v[a];
  }
}

template <int N, int E, typename T>
cudaError_t launch_interp(const DevConsts &c, const double *h_ops, const void *u, void *uf, cudaStream_t s) {
  constexpr int NFP = N * N, NU = N * NFP;
  constexpr size_t SMEM = 128 + al128(2 * N * 8) + al128(NU * NV * E * sizeof(T)) + 128;
  static_assert(SMEM <= SMEM_MAX && FR_BLK % E == 0, "configuration");
  const uint64_t ld = (uint64_t)c.ld;
  bool fresh = true;
  MapCache::Ent *ent = ((MapCache *)c.map_cache)->get(0, u, nullptr, nullptr, fresh);
  CUtensorMap &mU = ent->m[0];
  if (fresh && !encode3(&mU, sizeof(T) == 8, u, ld, NFP * NV, N, ld, (uint64_t)NFP * NV * ld, E, NFP * NV, N)) { ent->id = -1; return cudaErrorNotSupported; }
  auto kern = k_hex_interp_tma<N, E, T>;
  static DevFlags done;
  cudaError_t err = set_smem(kern, SMEM, done, c.dev);
  if (err != cudaSuccess) return err;
  kern<<<(unsigned)((c.Nel + E - 1) / E), N * N * E, SMEM, s>>>(mU, make_ops<N>(h_ops), c.ph, (T *)uf, c.ld, c.Nel);
  return cudaGetLastError();
}

// elements per CTA of this kernel: as the other kernels, except N = 7 where its small footprint allows 64-byte rows
template <int N>
struct EI {
  static constexpr int E = N == 7 ? 8 : Cfg<N, double>::E;
};

}  // namespace

cudaError_t hex_tma_interp(const DevConsts &c, const double *h_ops, const void *u, void *uf, cudaStream_t s) {
  switch (c.n) {
#define FR_CASE(NN) \
  case NN: return c.f64 ? launch_interp<NN, EI<NN>::E, double>(c, h_ops, u, uf, s) : launch_interp<NN, EI<NN>::E, float>(c, h_ops, u, uf, s);
    FR_CASE(2) FR_CASE(3) FR_CASE(4) FR_CASE(5) FR_CASE(6) FR_CASE(7)
#undef FR_CASE
    default: return cudaErrorNotSupported;
  }
}

}  // namespace fr
