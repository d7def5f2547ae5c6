// Register updates of the explicit time steppers (PAPER.md:247 RK4; Table 1 :263 Euler, RK4, DOPRI5): one streaming
// kernel forms up to two linear combinations of state-sized registers per pass.  Registers are [rows][ld] matrices in the
// storage precision; only the first nel columns of a row are touched (the pad columns of the caller's u stay as they are).
#include "fr_dev.hpp"

namespace fr {
namespace {

struct LinComb {
  int nin;
  const void *in[RK_MAX_IN];
  double a[RK_MAX_IN], b[RK_MAX_IN];  // out1 = sum a_i in_i,  out2 = sum b_i in_i  (zero coefficients: operand not read)
  void *out1, *out2;                  // either may be NULL; may alias an input (element-wise update)
};

template <typename T>
__global__ void __launch_bounds__(256) k_lincomb(const __grid_constant__ LinComb lc, int64_t rows, int64_t ld, int64_t nel) {
  const int64_t col = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (col >= nel) return;
  for (int64_t r = blockIdx.y; r < rows; r += gridDim.y) {
    const size_t o = (size_t)r * ld + col;
    double s1 = 0.0, s2 = 0.0;
#pragma unroll
    for (int i = 0; i < RK_MAX_IN; ++i) {
      if (i < lc.nin && (lc.a[i] != 0.0 || lc.b[i] != 0.0)) {
        const double v = (double)((const T *)lc.in[i])[o];
        s1 = fma(lc.a[i], v, s1);
        s2 = fma(lc.b[i], v, s2);
      }
    }
    if (lc.out1) ((T *)lc.out1)[o] = (T)s1;
    if (lc.out2) ((T *)lc.out2)[o] = (T)s2;
  }
}

// sum over the first nel columns of (x - y)^2, deterministic: one partial per CTA row chunk, then a single-CTA pass
template <typename T>
__global__ void __launch_bounds__(256) k_sqdiff_partial(const T *__restrict__ x, const T *__restrict__ y, int64_t rows, int64_t ld, int64_t nel,
                                                        double *__restrict__ part) {
  __shared__ double sh[256];
  double s = 0.0;
  const int64_t col0 = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  for (int64_t r = blockIdx.y; r < rows; r += gridDim.y)
    for (int64_t col = col0; col < nel; col += (int64_t)gridDim.x * blockDim.x) {
      const double d = (double)x[(size_t)r * ld + col] - (double)y[(size_t)r * ld + col];
      s = fma(d, d, s);
    }
  sh[threadIdx.x] = s;
  __syncthreads();
  for (int w = 128; w > 0; w >>= 1) {
    if ((int)threadIdx.x < w) sh[threadIdx.x] += sh[threadIdx.x + w];
    __syncthreads();
  }
  if (threadIdx.x == 0) part[(size_t)blockIdx.y * gridDim.x + blockIdx.x] = sh[0];
}

__global__ void __launch_bounds__(256) k_rms_final(const double *__restrict__ part, int n, double count, double *__restrict__ out) {
  __shared__ double sh[256];
  double s = 0.0;
  for (int i = threadIdx.x; i < n; i += 256) s += part[i];
  sh[threadIdx.x] = s;
  __syncthreads();
  for (int w = 128; w > 0; w >>= 1) {
    if ((int)threadIdx.x < w) sh[threadIdx.x] += sh[threadIdx.x + w];
    __syncthreads();
  }
  if (threadIdx.x == 0) *out = sqrt(sh[0] / count);
}

}  // namespace

cudaError_t rk_lincomb(bool f64, int64_t rows, int64_t ld, int64_t nel, int nin, const void *const *in, const double *a, const double *b,
                       void *out1, void *out2, cudaStream_t s) {
  if (nin < 1 || nin > RK_MAX_IN) return cudaErrorInvalidValue;
  LinComb lc{};
  lc.nin = nin;
  for (int i = 0; i < nin; ++i) { lc.in[i] = in[i]; lc.a[i] = a ? a[i] : 0.0; lc.b[i] = b ? b[i] : 0.0; }
  lc.out1 = out1; lc.out2 = out2;
  const int TB = 256;
  const unsigned gx = (unsigned)((nel + TB - 1) / TB);
  int64_t gy = (148 * 16 + gx - 1) / gx;  // about 16 CTAs per SM in total
  if (gy > rows) gy = rows;
  if (gy < 1) gy = 1;
  if (gy > 65535) gy = 65535;
  if (f64) k_lincomb<double><<<dim3(gx, (unsigned)gy), TB, 0, s>>>(lc, rows, ld, nel);
  else k_lincomb<float><<<dim3(gx, (unsigned)gy), TB, 0, s>>>(lc, rows, ld, nel);
  return cudaGetLastError();
}

cudaError_t rk_rms_diff(bool f64, int64_t rows, int64_t ld, int64_t nel, const void *x, const void *y, double *part, double *out,
                        cudaStream_t s) {
  const int TB = 256;
  unsigned gx = (unsigned)((nel + TB - 1) / TB);
  if (gx > 64) gx = 64;
  unsigned gy = (unsigned)(RK_MAX_PARTIALS / gx);
  if (gy > rows) gy = (unsigned)rows;
  if (gy < 1) gy = 1;
  if (f64) k_sqdiff_partial<double><<<dim3(gx, gy), TB, 0, s>>>((const double *)x, (const double *)y, rows, ld, nel, part);
  else k_sqdiff_partial<float><<<dim3(gx, gy), TB, 0, s>>>((const float *)x, (const float *)y, rows, ld, nel, part);
  k_rms_final<<<1, 256, 0, s>>>(part, (int)(gx * gy), (double)rows * (double)nel, out);
  return cudaGetLastError();
}

}  // namespace fr
