// 1-D factors of the tensor-product operators as a kernel parameter (constant bank).
#pragma once

namespace fr {

template <int N, typename R = double>
struct Ops1D {
  R D[N * N];    // D[i][m] = l_m'(xi_i)
  R Dh[N * N];   // D + gm lm^T - gp lp^T  (1-D form of M1 - M3 M2, Eq 44 :773; M2 holds n~ = -1 on the -1 face)
  R lm[N], lp[N];  // l_m(-1), l_m(+1)                    (M0, Eq 41)
  R gm[N], gp[N];  // div g of the -1 / +1 face point at node i (M3, M6)
};

__host__ __device__ constexpr int ipow(int b, int e) { return e == 0 ? 1 : b * ipow(b, e - 1); }

template <int N, typename R = double>
inline Ops1D<N, R> make_ops(const double *h) {  // h: D, Dh, lm, lp, gm, gp packed (TensorPlan::h_ops)
  Ops1D<N, R> o;
  const double *p = h;
  for (int i = 0; i < N * N; ++i) o.D[i] = (R)*p++;
  for (int i = 0; i < N * N; ++i) o.Dh[i] = (R)*p++;
  for (int i = 0; i < N; ++i) o.lm[i] = (R)*p++;
  for (int i = 0; i < N; ++i) o.lp[i] = (R)*p++;
  for (int i = 0; i < N; ++i) o.gm[i] = (R)*p++;
  for (int i = 0; i < N; ++i) o.gp[i] = (R)*p++;
  return o;
}

}  // namespace fr
