// Host operator builder: the constant operator matrices M0..M6 of PAPER.md:737-768 (Appendix A) from
// the nodal basis (:182) and the DG correction function (reading A5), in binary128, rounded once.
//
// Independent of oracle/: tensor elements are assembled from 1-D factors (Lagrange derivative matrix,
// end-point values, derivative of the Radau polynomials g_R = (P_p + P_{p+1})/2); triangles use a
// monomial Vandermonde with closed-form monomial integrals for the mass matrix.
#include <quadmath.h>

#include <cmath>
#include <stdexcept>

#include "fr_host.hpp"

namespace fr {
namespace {

typedef __float128 real;

void legendre(int n, real x, real &p, real &dp) {
  real p0 = 1, p1 = x, d0 = 0, d1 = 1;
  if (n == 0) { p = 1; dp = 0; return; }
  for (int k = 1; k < n; ++k) {
    real p2 = ((2 * k + 1) * x * p1 - k * p0) / (k + 1);
    real d2 = ((2 * k + 1) * (p1 + x * d1) - k * d0) / (k + 1);
    p0 = p1; p1 = p2; d0 = d1; d1 = d2;
  }
  p = p1; dp = d1;
}

// Gauss-Legendre points (ascending) and weights: Newton iteration on P_n
void gauss_legendre(int n, std::vector<real> &x, std::vector<real> &w) {
  x.resize(n); w.resize(n);
  for (int i = 0; i < n; ++i) {
    real xi = -cosq(M_PIq * (i + 1 - (real)0.25) / (n + (real)0.5));
    for (int it = 0; it < 200; ++it) {
      real p, dp; legendre(n, xi, p, dp);
      real dx = p / dp; xi -= dx;
      if (fabsq(dx) < 1e-33Q) break;
    }
    real p, dp; legendre(n, xi, p, dp);
    x[i] = xi; w[i] = 2 / ((1 - xi * xi) * dp * dp);
  }
  for (int i = 0; i < n / 2; ++i) {  // enforce exact symmetry
    real a = (x[n - 1 - i] - x[i]) / 2; x[i] = -a; x[n - 1 - i] = a;
    real b = (w[i] + w[n - 1 - i]) / 2; w[i] = w[n - 1 - i] = b;
  }
  if (n % 2) x[n / 2] = 0;
}

// 1-D Lagrange basis on `nodes` at x: L[j], dL[j]
void lagrange1d(const std::vector<real> &nodes, real x, std::vector<real> &L, std::vector<real> &dL) {
  int n = (int)nodes.size();
  L.assign(n, 1); dL.assign(n, 0);
  for (int j = 0; j < n; ++j) {
    for (int m = 0; m < n; ++m) if (m != j) L[j] *= (x - nodes[m]) / (nodes[j] - nodes[m]);
    for (int i = 0; i < n; ++i) {
      if (i == j) continue;
      real t = 1 / (nodes[j] - nodes[i]);
      for (int m = 0; m < n; ++m) if (m != j && m != i) t *= (x - nodes[m]) / (nodes[j] - nodes[m]);
      dL[j] += t;
    }
  }
}

void gauss_jordan(std::vector<real> &A, std::vector<real> &B, int n, int nb) {  // solves A X = B in place (B <- X)
  for (int c = 0; c < n; ++c) {
    int piv = c;
    for (int r = c + 1; r < n; ++r) if (fabsq(A[r * n + c]) > fabsq(A[piv * n + c])) piv = r;
    if (A[piv * n + c] == 0) throw std::runtime_error("singular Vandermonde / mass matrix");
    if (piv != c) {
      for (int k = 0; k < n; ++k) std::swap(A[c * n + k], A[piv * n + k]);
      for (int k = 0; k < nb; ++k) std::swap(B[c * nb + k], B[piv * nb + k]);
    }
    real d = A[c * n + c];
    for (int k = 0; k < n; ++k) A[c * n + k] /= d;
    for (int k = 0; k < nb; ++k) B[c * nb + k] /= d;
    for (int r = 0; r < n; ++r) {
      if (r == c) continue;
      real f = A[r * n + c];
      if (f == 0) continue;
      for (int k = 0; k < n; ++k) A[r * n + k] -= f * A[c * n + k];
      for (int k = 0; k < nb; ++k) B[r * nb + k] -= f * B[c * nb + k];
    }
  }
}

real ipow(real x, int e) { real r = 1; for (int i = 0; i < e; ++i) r *= x; return r; }
real fact(int k) { real r = 1; for (int i = 2; i <= k; ++i) r *= i; return r; }
real binom(int a, int i) { return fact(a) / (fact(i) * fact(a - i)); }

// integral of x^a y^b over the reference triangle (-1,-1),(1,-1),(-1,1):
// x = 2r-1, y = 2s-1 on the unit triangle, dA = 4 dr ds, int r^i s^j = i! j! / (i+j+2)!
real tri_monomial_integral(int a, int b) {
  real s = 0;
  for (int i = 0; i <= a; ++i)
    for (int j = 0; j <= b; ++j) {
      real c = binom(a, i) * ipow(2, i) * (((a - i) % 2) ? -1 : 1) * binom(b, j) * ipow(2, j) * (((b - j) % 2) ? -1 : 1);
      s += c * fact(i) * fact(j) / fact(i + j + 2);
    }
  return 4 * s;
}

// Nodal basis on an arbitrary point set of the triangle, monomial Vandermonde
struct TriBasis {
  int p, N;
  std::vector<int> ea, eb;
  std::vector<real> c;  // l_sigma(x) = sum_m psi_m(x) c[m][sigma]
  TriBasis(int p_, const std::vector<real> &pts) : p(p_) {
    for (int b = 0; b <= p; ++b) for (int a = 0; a <= p - b; ++a) { ea.push_back(a); eb.push_back(b); }
    N = (int)ea.size();
    std::vector<real> V(N * N);
    for (int s = 0; s < N; ++s) for (int m = 0; m < N; ++m) V[s * N + m] = ipow(pts[2 * s], ea[m]) * ipow(pts[2 * s + 1], eb[m]);
    c.assign(N * N, 0);
    for (int i = 0; i < N; ++i) c[i * N + i] = 1;
    gauss_jordan(V, c, N, N);  // V c = I
  }
  void eval(real x, real y, std::vector<real> &L, std::vector<real> &dLx, std::vector<real> &dLy) const {
    L.assign(N, 0); dLx.assign(N, 0); dLy.assign(N, 0);
    for (int m = 0; m < N; ++m) {
      real v = ipow(x, ea[m]) * ipow(y, eb[m]);
      real vx = ea[m] ? ea[m] * ipow(x, ea[m] - 1) * ipow(y, eb[m]) : (real)0;
      real vy = eb[m] ? eb[m] * ipow(x, ea[m]) * ipow(y, eb[m] - 1) : (real)0;
      for (int s = 0; s < N; ++s) { L[s] += v * c[m * N + s]; dLx[s] += vx * c[m * N + s]; dLy[s] += vy * c[m * N + s]; }
    }
  }
  // exact mass matrix of the nodal basis: c^T G c with G the monomial Gram matrix
  std::vector<real> mass() const {
    std::vector<real> G(N * N), T(N * N, 0), Mm(N * N, 0);
    for (int a = 0; a < N; ++a) for (int b = 0; b < N; ++b) G[a * N + b] = tri_monomial_integral(ea[a] + ea[b], eb[a] + eb[b]);
    for (int a = 0; a < N; ++a) for (int s = 0; s < N; ++s) { real t = 0; for (int b = 0; b < N; ++b) t += G[a * N + b] * c[b * N + s]; T[a * N + s] = t; }
    for (int r = 0; r < N; ++r) for (int s = 0; s < N; ++s) { real t = 0; for (int a = 0; a < N; ++a) t += c[a * N + r] * T[a * N + s]; Mm[r * N + s] = t; }
    return Mm;
  }
};

std::vector<double> round_to_double(const std::vector<real> &a) {
  std::vector<double> r(a.size());
  for (size_t i = 0; i < a.size(); ++i) r[i] = (double)a[i];
  return r;
}
std::vector<long double> round_to_ld(const std::vector<real> &a) {
  std::vector<long double> r(a.size());
  for (size_t i = 0; i < a.size(); ++i) r[i] = (long double)a[i];
  return r;
}

int ipowi(int b, int e) { int r = 1; for (int i = 0; i < e; ++i) r *= b; return r; }

}  // namespace

void build_ref_ops(int etype, int p, int p_g, int correction, RefOps &o) {
  if (p < 0 || p > 12) throw std::runtime_error("polynomial order p out of range [0,12]");
  if (correction != FR_CORR_DG && correction != FR_CORR_SD && correction != FR_CORR_HU) throw std::runtime_error("unknown correction function");
  if (correction != FR_CORR_DG && etype == FR_TRI) throw std::runtime_error("SD / HU correction functions are available on quadrilaterals and hexahedra only");
  if (correction == FR_CORR_HU && p < 1) throw std::runtime_error("the HU correction function needs p >= 1");
  if (p_g < 1 || p_g > 8) throw std::runtime_error("geometry degree p_g out of range [1,8]");
  o = RefOps();
  o.etype = etype; o.p = p; o.n = p + 1; o.p_g = p_g;
  const int n = p + 1;
  const int nd = (etype == FR_HEX) ? 3 : 2;
  o.nd = nd;
  std::vector<real> g, w;
  gauss_legendre(n, g, w);
  std::vector<real> xu, xf, nf, wu, wf;
  std::vector<real> M0, M1, M2, M3, M4, M6;

  if (etype == FR_QUAD || etype == FR_HEX) {
    const int Nu = ipowi(n, nd), nfp = ipowi(n, nd - 1), Nf = 2 * nd * nfp;
    o.Nu = Nu; o.Nf = Nf; o.nfaces = 2 * nd; o.nfp = nfp;
    // 1-D factors
    std::vector<real> D(n * n), lm(n), lp(n), gm(n), gp(n), L, dL;
    for (int i = 0; i < n; ++i) { lagrange1d(g, g[i], L, dL); for (int j = 0; j < n; ++j) D[i * n + j] = dL[j]; }
    lagrange1d(g, -1, lm, dL);
    lagrange1d(g, 1, lp, dL);
    // One-parameter family of energy-stable correction functions of the paper's ref [10] ("DG, SD, and HU as
    // defined in [10]"; reading A23):  g_R = {P_p + (eta P_{p-1} + P_{p+1}) / (1 + eta)} / 2,  eta = c (2p+1) (a_p p!)^2 / 2,
    // a_p = (2p)! / (2^p (p!)^2);  c = 0 (DG: g_R = Radau, A5),  c_SD = 2p / ((2p+1)(p+1)(a_p p!)^2),
    // c_HU = 2(p+1) / ((2p+1) p (a_p p!)^2).  The -1 face uses g_R'(-xi) (outward-normal convention).
    real eta = 0;
    if (correction != FR_CORR_DG) {
      const real ap = fact(2 * p) / (ipow(2, p) * fact(p) * fact(p));
      const real apf2 = (ap * fact(p)) * (ap * fact(p));
      const real c = correction == FR_CORR_SD ? (real)(2 * p) / ((2 * p + 1) * (p + 1) * apf2) : (real)(2 * (p + 1)) / ((2 * p + 1) * p * apf2);
      eta = c * (2 * p + 1) * apf2 / 2;
    }
    auto dgr = [&](real x) {
      real a, da, b, db, m = 0, dm = 0;
      legendre(p, x, a, da); legendre(p + 1, x, b, db);
      if (p >= 1) legendre(p - 1, x, m, dm);
      return (da + (eta * dm + db) / (1 + eta)) / 2;
    };
    for (int i = 0; i < n; ++i) { gp[i] = dgr(g[i]); gm[i] = dgr(-g[i]); }
    std::vector<real> Dh(n * n);
    for (int i = 0; i < n; ++i) for (int j = 0; j < n; ++j) Dh[i * n + j] = D[i * n + j] + gm[i] * lm[j] - gp[i] * lp[j];  // M2 carries the reference normal: -1 on the -1 face
    o.D1 = round_to_double(D); o.lm = round_to_double(lm); o.lp = round_to_double(lp);
    o.gm = round_to_double(gm); o.gp = round_to_double(gp); o.Dhat = round_to_double(Dh);
    // point sets
    xu.assign(Nu * nd, 0); wu.assign(Nu, 1);
    auto idx_of = [&](int rho, int d) { return (rho / ipowi(n, d)) % n; };
    for (int r = 0; r < Nu; ++r) for (int d = 0; d < nd; ++d) { xu[r * nd + d] = g[idx_of(r, d)]; wu[r] *= w[idx_of(r, d)]; }
    xf.assign(Nf * nd, 0); nf.assign(Nf * nd, 0); wf.assign(Nf, 1);
    std::vector<int> fidx(Nf * nd, -1);  // tensor index of the flux point in the non-normal directions
    for (int d = 0; d < nd; ++d) for (int s = 0; s < 2; ++s) for (int k = 0; k < nfp; ++k) {
      int sig = (2 * d + s) * nfp + k;
      xf[sig * nd + d] = s ? 1 : -1; nf[sig * nd + d] = s ? 1 : -1;
      int m = 0;
      for (int dd = 0; dd < nd; ++dd) {
        if (dd == d) continue;
        int i = (k / ipowi(n, m)) % n; ++m;
        xf[sig * nd + dd] = g[i]; wf[sig] *= w[i]; fidx[sig * nd + dd] = i;
      }
    }
    // dense operators from the 1-D factors
    M0.assign(Nf * Nu, 0); M3.assign(Nu * Nf, 0);
    for (int sig = 0; sig < Nf; ++sig) {
      int d = (sig / nfp) / 2, s = (sig / nfp) % 2;
      for (int r = 0; r < Nu; ++r) {
        bool on_line = true;
        for (int dd = 0; dd < nd; ++dd) if (dd != d && idx_of(r, dd) != fidx[sig * nd + dd]) on_line = false;
        if (!on_line) continue;
        M0[sig * Nu + r] = s ? lp[idx_of(r, d)] : lm[idx_of(r, d)];
        M3[r * Nf + sig] = s ? gp[idx_of(r, d)] : gm[idx_of(r, d)];
      }
    }
    M4.assign(nd * Nu * Nu, 0); M1.assign(Nu * nd * Nu, 0);
    for (int d = 0; d < nd; ++d) for (int s = 0; s < Nu; ++s) for (int r = 0; r < Nu; ++r) {
      bool on_line = true;
      for (int dd = 0; dd < nd; ++dd) if (dd != d && idx_of(r, dd) != idx_of(s, dd)) on_line = false;
      if (!on_line) continue;
      real v = D[idx_of(s, d) * n + idx_of(r, d)];  // d_d l_r at x_s
      M4[(d * Nu + s) * Nu + r] = v;
      M1[s * (nd * Nu) + d * Nu + r] = v;
    }
  } else if (etype == FR_TRI) {
    const int Nu = n * (n + 1) / 2, Nf = 3 * n;
    o.Nu = Nu; o.Nf = Nf; o.nfaces = 3; o.nfp = n;
    for (int j = 0; j <= p; ++j) for (int i = 0; i <= p - j; ++i) {  // barycentric lattice (A6)
      xu.push_back(-1 + 2 * (real)(i + 1) / (p + 3)); xu.push_back(-1 + 2 * (real)(j + 1) / (p + 3));
    }
    const real r2 = sqrtq((real)2);
    const real vx[3] = {-1, 1, -1}, vy[3] = {-1, -1, 1};
    const real nx[3] = {0, 1 / r2, -1}, ny[3] = {-1, 1 / r2, 0}, sc[3] = {1, r2, 1};
    for (int k = 0; k < 3; ++k) for (int i = 0; i < n; ++i) {
      int k1 = (k + 1) % 3;
      xf.push_back((vx[k] * (1 - g[i]) + vx[k1] * (1 + g[i])) / 2);
      xf.push_back((vy[k] * (1 - g[i]) + vy[k1] * (1 + g[i])) / 2);
      nf.push_back(nx[k]); nf.push_back(ny[k]); wf.push_back(w[i] * sc[k]);
    }
    TriBasis B(p, xu);
    std::vector<real> L, dx, dy;
    M0.assign(Nf * Nu, 0);
    for (int s = 0; s < Nf; ++s) { B.eval(xf[2 * s], xf[2 * s + 1], L, dx, dy); for (int r = 0; r < Nu; ++r) M0[s * Nu + r] = L[r]; }
    M4.assign(2 * Nu * Nu, 0); M1.assign(Nu * 2 * Nu, 0);
    for (int s = 0; s < Nu; ++s) {
      B.eval(xu[2 * s], xu[2 * s + 1], L, dx, dy);
      for (int r = 0; r < Nu; ++r) {
        M4[(0 * Nu + s) * Nu + r] = dx[r]; M4[(1 * Nu + s) * Nu + r] = dy[r];
        M1[s * 2 * Nu + r] = dx[r]; M1[s * 2 * Nu + Nu + r] = dy[r];
      }
    }
    // DG correction (A5): M3 = Mass^-1 M0^T diag(w^f)
    std::vector<real> Mm = B.mass();
    M3.assign(Nu * Nf, 0);
    for (int r = 0; r < Nu; ++r) for (int s = 0; s < Nf; ++s) M3[r * Nf + s] = M0[s * Nu + r] * wf[s];
    wu.assign(Nu, 0);
    for (int r = 0; r < Nu; ++r) for (int s = 0; s < Nu; ++s) wu[r] += Mm[r * Nu + s];  // integral of l_r = sum_s M_rs
    gauss_jordan(Mm, M3, Nu, Nf);
  } else {
    throw std::runtime_error("unknown element type");
  }
  const int Nu = o.Nu, Nf = o.Nf;
  M2.assign(Nf * nd * Nu, 0); M6.assign(nd * Nu * Nf, 0);
  for (int s = 0; s < Nf; ++s) for (int d = 0; d < nd; ++d) for (int r = 0; r < Nu; ++r) {
    M2[s * (nd * Nu) + d * Nu + r] = M0[s * Nu + r] * nf[s * nd + d];   // :768
    M6[(d * Nu + r) * Nf + s] = nf[s * nd + d] * M3[r * Nf + s];        // :749 (A1)
  }
  // fused operators (Eq 42 :756, Eq 44 :773) in binary128
  std::vector<real> M46(nd * Nu * Nu), M132(Nu * nd * Nu);
  for (int r = 0; r < nd * Nu; ++r) for (int c = 0; c < Nu; ++c) {
    real t = M4[r * Nu + c];
    for (int s = 0; s < Nf; ++s) t -= M6[r * Nf + s] * M0[s * Nu + c];
    M46[r * Nu + c] = t;
  }
  for (int r = 0; r < Nu; ++r) for (int c = 0; c < nd * Nu; ++c) {
    real t = M1[r * nd * Nu + c];
    for (int s = 0; s < Nf; ++s) t -= M3[r * Nf + s] * M2[s * nd * Nu + c];
    M132[r * nd * Nu + c] = t;
  }
  o.M[0] = round_to_double(M0); o.rows[0] = Nf; o.cols[0] = Nu;
  o.M[1] = round_to_double(M1); o.rows[1] = Nu; o.cols[1] = nd * Nu;
  o.M[2] = round_to_double(M2); o.rows[2] = Nf; o.cols[2] = nd * Nu;
  o.M[3] = round_to_double(M3); o.rows[3] = Nu; o.cols[3] = Nf;
  o.M[4] = round_to_double(M4); o.rows[4] = nd * Nu; o.cols[4] = Nu;
  o.M[5].assign((size_t)nd * Nf * nd * Nu, 0.0); o.rows[5] = nd * Nf; o.cols[5] = nd * Nu;  // diag(M0) :760
  for (int d = 0; d < nd; ++d) for (int s = 0; s < Nf; ++s) for (int r = 0; r < Nu; ++r)
    o.M[5][(size_t)(d * Nf + s) * nd * Nu + d * Nu + r] = (double)M0[s * Nu + r];
  o.M[6] = round_to_double(M6); o.rows[6] = nd * Nu; o.cols[6] = Nf;
  o.M46 = round_to_double(M46); o.M132 = round_to_double(M132);
  o.xu = round_to_ld(xu); o.xf = round_to_ld(xf); o.nf = round_to_ld(nf);
  o.wu = round_to_double(wu); o.wf = round_to_double(wf);

  // geometry basis of degree p_g on the equispaced lattice, evaluated at solution and flux points
  auto geom_eval = [&](const std::vector<real> &pts, int npts, std::vector<long double> &G, std::vector<long double> &dG) {
    if (etype == FR_TRI) {
      std::vector<real> nodes;
      for (int j = 0; j <= p_g; ++j) for (int i = 0; i <= p_g - j; ++i) { nodes.push_back(-1 + 2 * (real)i / p_g); nodes.push_back(-1 + 2 * (real)j / p_g); }
      TriBasis B(p_g, nodes);
      o.Nn = B.N;
      G.assign((size_t)npts * B.N, 0); dG.assign((size_t)2 * npts * B.N, 0);
      std::vector<real> L, dx, dy;
      for (int s = 0; s < npts; ++s) {
        B.eval(pts[2 * s], pts[2 * s + 1], L, dx, dy);
        for (int k = 0; k < B.N; ++k) { G[(size_t)s * B.N + k] = (long double)L[k]; dG[(size_t)(0 * npts + s) * B.N + k] = (long double)dx[k]; dG[(size_t)(1 * npts + s) * B.N + k] = (long double)dy[k]; }
      }
    } else {
      int m = p_g + 1, Nn = ipowi(m, nd);
      o.Nn = Nn;
      std::vector<real> nodes(m);
      for (int i = 0; i < m; ++i) nodes[i] = -1 + 2 * (real)i / p_g;
      G.assign((size_t)npts * Nn, 0); dG.assign((size_t)nd * npts * Nn, 0);
      std::vector<real> L[3], dL[3];
      for (int s = 0; s < npts; ++s) {
        for (int d = 0; d < nd; ++d) lagrange1d(nodes, pts[s * nd + d], L[d], dL[d]);
        for (int k = 0; k < Nn; ++k) {
          real v = 1;
          for (int d = 0; d < nd; ++d) v *= L[d][(k / ipowi(m, d)) % m];
          G[(size_t)s * Nn + k] = (long double)v;
          for (int dd = 0; dd < nd; ++dd) {
            real t = 1;
            for (int d = 0; d < nd; ++d) t *= (d == dd ? dL[d] : L[d])[(k / ipowi(m, d)) % m];
            dG[(size_t)(dd * npts + s) * Nn + k] = (long double)t;
          }
        }
      }
    }
  };
  geom_eval(xu, Nu, o.Gu, o.dGu);
  geom_eval(xf, Nf, o.Gf, o.dGf);
}

}  // namespace fr
