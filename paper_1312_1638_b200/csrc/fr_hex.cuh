// Fused hexahedral kernels, "z-slab streaming": a CTA owns E consecutive elements; thread (e, i, j) owns the
// column of n solution points (i, j, k = 0..n-1) of element e and walks it slice by slice.  Contractions
// along z stay in registers, contractions along x and y go through one shared-memory slice, so the
// transformed flux F~ (Eq 12) never reaches HBM: parts (4), (6), (7) of the north_star are one kernel.
// Every global access is a row segment of E consecutive elements (E*8 bytes, 128 B at E = 16).
// Included inside fr_tensor.cu's anonymous namespace (needs Ops1D, ipow).

// F~ = S f(u, q) at one point (Eq 12 :214 with Eq 20-24)
template <bool NS>
__device__ __forceinline__ void point_tflux(const double *uu, const double (*qq)[5], const double (*S)[3], const Phys &ph,
                                            double (*F)[5]) {
  double f[3][5], v[3], p;
  inviscid_flux<3>(uu, ph.gamma, f, v, p);
  if (NS) subtract_viscous_flux<3>(uu, qq, v, ph, f);
#pragma unroll
  for (int i = 0; i < 3; ++i)
#pragma unroll
    for (int a = 0; a < 5; ++a) F[i][a] = fma(S[i][0], f[0][a], fma(S[i][1], f[1][a], S[i][2] * f[2][a]));
}

// rhs = -(1/J) {(M1 - M3 M2) F~ + M3 D~},  F~ = S f(U, Q)   (Eq 12, 18, 19 / Eq 44)
// u [NU][5][ld] (T), q [3][NU][5][ld], smat [9][NU][ld], rcpj [NU][ld], dt = D~ [NF][5][ld], rhs like u.
template <int N, int E, bool NS, typename T>
__global__ void __launch_bounds__(N *N *E) k_hex_fluxdiv(Ops1D<N> op, Phys ph, const T *__restrict__ u, const double *__restrict__ q,
                                                         const double *__restrict__ smat, const double *__restrict__ rcpj,
                                                         const double *__restrict__ dt, T *__restrict__ rhs, int64_t ld, int64_t Nel) {
  constexpr int NV = 5, NFP = N * N, NU = N * N * N;
  extern __shared__ double smem[];
  double *sDh = smem;                 // [N*N]
  double *sF = smem + N * N;          // [2 buffers][2 directions][NV][NFP][E]
  const int el = threadIdx.x, ij = threadIdx.y, i = ij % N, j = ij / N;
  const int64_t e = (int64_t)blockIdx.x * E + el;
  const bool act = e < Nel;
  const size_t ncols = (size_t)NV * ld;
  if (ij == 0 && el < N * N) sDh[el] = op.Dh[el];
  if (N * N > E && ij == 1 && el + E < N * N) sDh[el + E] = op.Dh[el + E];
  if (N * N > 2 * E && ij == 2) for (int t = el + 2 * E; t < N * N; t += E) sDh[t] = op.Dh[t];

  double acc[N][NV];
#pragma unroll
  for (int k = 0; k < N; ++k)
#pragma unroll
    for (int a = 0; a < NV; ++a) acc[k][a] = 0.0;

#pragma unroll
  for (int k = 0; k < N; ++k) {
    const int r = ij + NFP * k;
    double F[3][NV];
    if (act) {
      double uu[NV], qq[3][NV], S[3][3];
#pragma unroll
      for (int a = 0; a < NV; ++a) uu[a] = (double)u[((size_t)r * NV + a) * ld + e];
      if (NS) {
#pragma unroll
        for (int n = 0; n < 3; ++n)
#pragma unroll
          for (int a = 0; a < NV; ++a) qq[n][a] = q[(((size_t)n * NU + r) * NV + a) * ld + e];
      }
#pragma unroll
      for (int a = 0; a < 3; ++a)
#pragma unroll
        for (int b = 0; b < 3; ++b) S[a][b] = smat[((size_t)(a * 3 + b) * NU + r) * ld + e];
      point_tflux<NS>(uu, qq, S, ph, F);
    } else {
#pragma unroll
      for (int d = 0; d < 3; ++d)
#pragma unroll
        for (int a = 0; a < NV; ++a) F[d][a] = 0.0;
    }
    double *buf = sF + (k & 1) * (2 * NV * NFP * E);
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
  const double gmi = op.gm[i], gpi = op.gp[i], gmj = op.gm[j], gpj = op.gp[j];
#pragma unroll
  for (int k = 0; k < N; ++k) {
    const int r = ij + NFP * k;
    const double rj = rcpj[(size_t)r * ld + e];
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

// Q = J^-T {M4 U + M6 (C - U^f)}  (Eq 9-10 / Eq 42) for all variables of a column of points.
// u [NU][5][ld] (T), jump = C - U^f [NF][5][ld], q out [3][NU][5][ld].
template <int N, int E, typename T>
__global__ void __launch_bounds__(N *N *E) k_hex_grad(Ops1D<N> op, const T *__restrict__ u, const double *__restrict__ jump,
                                                      const double *__restrict__ smat, const double *__restrict__ rcpj,
                                                      double *__restrict__ q, int64_t ld, int64_t Nel) {
  constexpr int NV = 5, NFP = N * N, NU = N * N * N;
  extern __shared__ double smem[];
  double *sD = smem;            // [N*N]
  double *sU = smem + N * N;    // [2 buffers][NV][NFP][E]
  const int el = threadIdx.x, ij = threadIdx.y, i = ij % N, j = ij / N;
  const int64_t e = (int64_t)blockIdx.x * E + el;
  const bool act = e < Nel;
  for (int t = ij * E + el; t < N * N; t += NFP * E) sD[t] = op.D[t];

  double ucol[N][NV], jzm[NV], jzp[NV];
#pragma unroll
  for (int k = 0; k < N; ++k)
#pragma unroll
    for (int a = 0; a < NV; ++a) ucol[k][a] = act ? (double)u[((size_t)(ij + NFP * k) * NV + a) * ld + e] : 0.0;
#pragma unroll
  for (int a = 0; a < NV; ++a) {
    jzm[a] = act ? jump[((size_t)(4 * NFP + ij) * NV + a) * ld + e] : 0.0;
    jzp[a] = act ? jump[((size_t)(5 * NFP + ij) * NV + a) * ld + e] : 0.0;
  }
  const double gmi = op.gm[i], gpi = op.gp[i], gmj = op.gm[j], gpj = op.gp[j];

#pragma unroll
  for (int k = 0; k < N; ++k) {
    const int r = ij + NFP * k;
    double *buf = sU + (k & 1) * (NV * NFP * E);
#pragma unroll
    for (int a = 0; a < NV; ++a) buf[(a * NFP + ij) * E + el] = ucol[k][a];
    __syncthreads();
    if (!act) continue;
    double S[3][3];
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
      for (int b = 0; b < 3; ++b) S[a][b] = smat[((size_t)(a * 3 + b) * NU + r) * ld + e];
    const double rj = rcpj[(size_t)r * ld + e];
    const int fx = j + N * k, fy = i + N * k;
#pragma unroll
    for (int a = 0; a < NV; ++a) {
      // M6 = n~ (x) M3 (A1): the reference normal is -1 on the -1 faces
      double qx = fma(gpi, jump[((size_t)(1 * NFP + fx) * NV + a) * ld + e], -gmi * jump[((size_t)(0 * NFP + fx) * NV + a) * ld + e]);
      double qy = fma(gpj, jump[((size_t)(3 * NFP + fy) * NV + a) * ld + e], -gmj * jump[((size_t)(2 * NFP + fy) * NV + a) * ld + e]);
      double qz = fma(op.gp[k], jzp[a], -op.gm[k] * jzm[a]);
#pragma unroll
      for (int m = 0; m < N; ++m) {
        qx = fma(sD[i * N + m], buf[(a * NFP + j * N + m) * E + el], qx);
        qy = fma(sD[j * N + m], buf[(a * NFP + m * N + i) * E + el], qy);
        qz = fma(op.D[k * N + m], ucol[m][a], qz);
      }
#pragma unroll
      for (int n = 0; n < 3; ++n)
        q[(((size_t)n * NU + r) * NV + a) * ld + e] = rj * fma(S[0][n], qx, fma(S[1][n], qy, S[2][n] * qz));
    }
  }
}
