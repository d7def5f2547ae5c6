// Mesh setup: metric terms at the solution points, physical normals at the flux points, and the
// flux-point lookup tables (PAPER.md:151-160 Jacobians, :216 S = J*J^-1, :223 Eq 14, :194 lookup table,
// :693 iteration order).  Host code, long double geometry, OpenMP over elements.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <numeric>
#include <parallel/algorithm>

#include "fr_host.hpp"

namespace fr {
namespace {

// x[i] and Jm[i][j] = dx_i/dxi_j at one point from the geometry basis rows G[Nn], dG[nd][npts][Nn]
inline void eval_point(int nd, int Nn, const double *X, const long double *G, const long double *dG, size_t dstride,
                       long double *x, long double Jm[3][3]) {
  for (int i = 0; i < nd; ++i) {
    long double s = 0;
    for (int k = 0; k < Nn; ++k) s += G[k] * (long double)X[k * nd + i];
    x[i] = s;
    for (int j = 0; j < nd; ++j) {
      long double t = 0;
      const long double *g = dG + j * dstride;
      for (int k = 0; k < Nn; ++k) t += g[k] * (long double)X[k * nd + i];
      Jm[i][j] = t;
    }
  }
}

// S = det(J) * J^-1 (adjugate), S[i][n] = J * dxi_i/dx_n; returns det J
inline long double adjugate(int nd, const long double Jm[3][3], long double S[3][3]) {
  if (nd == 2) {
    S[0][0] = Jm[1][1]; S[0][1] = -Jm[0][1];
    S[1][0] = -Jm[1][0]; S[1][1] = Jm[0][0];
    return Jm[0][0] * Jm[1][1] - Jm[0][1] * Jm[1][0];
  }
  for (int i = 0; i < 3; ++i)
    for (int n = 0; n < 3; ++n) {
      int a0 = (n + 1) % 3, a1 = (n + 2) % 3, b0 = (i + 1) % 3, b1 = (i + 2) % 3;
      S[i][n] = Jm[a0][b0] * Jm[a1][b1] - Jm[a0][b1] * Jm[a1][b0];
    }
  return Jm[0][0] * S[0][0] + Jm[0][1] * S[1][0] + Jm[0][2] * S[2][0];
}

}  // namespace

int build_mesh_consts(const MeshInput &in, const RefOps &ops, int64_t ld, int pair_block, MeshConsts &out, std::string &err,
                      bool standalone) {
  const int nd = in.nd, Nu = ops.Nu, Nf = ops.Nf, Nn = ops.Nn, nfp = ops.nfp;
  const int64_t Nel = in.Nel;
  out = MeshConsts();
  out.Nel = Nel; out.ld = ld;
  out.xu.assign((size_t)Nu * Nel * nd, 0.0);
  out.smat.assign((size_t)nd * nd * Nu * ld, 0.0);
  out.rcpj.assign((size_t)Nu * ld, 1.0);
  std::vector<double> xf((size_t)Nf * Nel * nd);
  out.fp_n.assign((size_t)nd * Nf * ld, 0.0);
  out.fp_Jn.assign((size_t)Nf * ld, 0.0);
  out.fp_pe.assign((size_t)Nf * ld, 0);
  out.fp_ps.assign((size_t)Nf * ld, 0);
  int bad = 0, nonaffine = 0;
#pragma omp parallel for schedule(static) reduction(+ : bad, nonaffine)
  for (int64_t e = 0; e < Nel; ++e) {
    const double *X = in.nodes.data() + (size_t)e * Nn * nd;
    long double x[3], Jm[3][3], S[3][3], S0[3][3];
    for (int r = 0; r < Nu; ++r) {
      eval_point(nd, Nn, X, &ops.Gu[(size_t)r * Nn], &ops.dGu[(size_t)r * Nn], (size_t)Nu * Nn, x, Jm);
      long double det = adjugate(nd, Jm, S);
      if (!(det > 0)) ++bad;
      for (int i = 0; i < nd; ++i) out.xu[((size_t)r * Nel + e) * nd + i] = (double)x[i];
      for (int i = 0; i < nd; ++i)
        for (int n = 0; n < nd; ++n) {
          out.smat[((size_t)(i * nd + n) * Nu + r) * ld + e] = (double)S[i][n];
          if (r == 0) S0[i][n] = S[i][n];
          else if (fabsl(S[i][n] - S0[i][n]) > 1e-13L * (fabsl(S0[i][n]) + fabsl(det))) ++nonaffine;
        }
      out.rcpj[(size_t)r * ld + e] = (double)(1.0L / det);
    }
    for (int s = 0; s < Nf; ++s) {
      eval_point(nd, Nn, X, &ops.Gf[(size_t)s * Nn], &ops.dGf[(size_t)s * Nn], (size_t)Nf * Nn, x, Jm);
      long double det = adjugate(nd, Jm, S);
      if (!(det > 0)) ++bad;
      long double v[3] = {0, 0, 0}, mag = 0;  // (S^T n~)_n = sum_i S[i][n] n~_i   (Eq 14, A15)
      for (int n = 0; n < nd; ++n) {
        for (int i = 0; i < nd; ++i) v[n] += S[i][n] * ops.nf[(size_t)s * nd + i];
        mag += v[n] * v[n];
      }
      mag = sqrtl(mag);
      for (int n = 0; n < nd; ++n) {
        xf[((size_t)s * Nel + e) * nd + n] = (double)x[n];
        out.fp_n[((size_t)n * Nf + s) * ld + e] = (double)(v[n] / mag);
      }
      out.fp_Jn[(size_t)s * ld + e] = (double)mag;
    }
  }
  if (bad) { err = "non-positive Jacobian determinant at " + std::to_string(bad) + " points"; return FR_EMESH; }
  out.affine = (nonaffine == 0);

  // ---- flux-point pairing by physical coordinates (PAPER.md:182 co-location, :194 lookup table) ----
  const int64_t nif = (int64_t)in.ifaces.size() / 4, nb = (int64_t)in.bfaces.size() / 3;
  std::vector<int32_t> cover((size_t)Nf * Nel, 0);
  struct Pair { int32_t Ls, Le, Rs, Re; };
  std::vector<Pair> pairs((size_t)nif * nfp);
  int unmatched = 0, range = 0;
#pragma omp parallel for schedule(static) reduction(+ : unmatched, range)
  for (int64_t f = 0; f < nif; ++f) {
    int32_t eL = in.ifaces[4 * f], fL = in.ifaces[4 * f + 1], eR = in.ifaces[4 * f + 2], fR = in.ifaces[4 * f + 3];
    if (eL < 0 || eL >= Nel || eR < 0 || eR >= Nel || fL < 0 || fL >= ops.nfaces || fR < 0 || fR >= ops.nfaces) { ++range; continue; }
    // face size for the tolerance
    double h2 = 0;
    for (int n = 0; n < nd; ++n) {
      double d = xf[((size_t)(fL * nfp) * Nel + eL) * nd + n] - xf[((size_t)(fL * nfp + nfp - 1) * Nel + eL) * nd + n];
      h2 += d * d;
    }
    double tol2 = 1e-18 * (h2 > 0 ? h2 : 1.0) + 1e-24;
    unsigned long long used = 0;
    for (int k = 0; k < nfp; ++k) {
      int sL = fL * nfp + k, best = -1;
      double bd = 1e300;
      for (int m = 0; m < nfp; ++m) {
        int sR = fR * nfp + m;
        double d2 = 0;
        for (int n = 0; n < nd; ++n) {
          double d = xf[((size_t)sL * Nel + eL) * nd + n] - (xf[((size_t)sR * Nel + eR) * nd + n] + in.shifts[(size_t)f * nd + n]);
          d2 += d * d;
        }
        if (d2 < bd) { bd = d2; best = m; }
      }
      if (!(bd <= tol2) || (nfp <= 64 && ((used >> best) & 1ull))) ++unmatched;
      if (nfp <= 64) used |= 1ull << best;
      pairs[(size_t)f * nfp + k] = {sL, eL, fR * nfp + best, eR};
    }
  }
  if (range) { err = "interface list references an element or face out of range"; return FR_EINVAL; }
  if (unmatched) { err = "unmatched flux-point pairs: " + std::to_string(unmatched); return FR_EMESH; }
  for (auto &pr : pairs) { cover[(size_t)pr.Ls * Nel + pr.Le]++; cover[(size_t)pr.Rs * Nel + pr.Re]++; }
  for (int64_t b = 0; b < nb; ++b) {
    int32_t e = in.bfaces[3 * b], f = in.bfaces[3 * b + 1], id = in.bfaces[3 * b + 2];
    if (e < 0 || e >= Nel || f < 0 || f >= ops.nfaces) { err = "boundary face out of range"; return FR_EINVAL; }
    if (id < 0 || id >= (int32_t)in.bcs.size()) { err = "boundary face references an undefined bc_id"; return FR_EINVAL; }
    for (int k = 0; k < nfp; ++k) cover[(size_t)(f * nfp + k) * Nel + e]++;
  }
  int64_t badcover = 0;
  for (auto c : cover) if (c != 1) ++badcover;
  if (badcover && standalone) { err = "flux points not covered exactly once by interfaces + boundary faces: " + std::to_string(badcover); return FR_EMESH; }

  // iteration order: sort by the L flux point (sigma major, element minor) so that consecutive threads
  // read consecutive elements of one row.  With element-blocked flux-point arrays (pair_block > 0
  // elements per block) the element block comes first, so that consecutive warps stay inside one block's rows.
  std::vector<int64_t> order(pairs.size());
  std::iota(order.begin(), order.end(), 0);
  auto key = [&](const Pair &pr) {
    if (pair_block <= 0) return (int64_t)pr.Ls * Nel + pr.Le;
    return ((int64_t)(pr.Le / pair_block) * Nf + pr.Ls) * pair_block + pr.Le % pair_block;
  };
  __gnu_parallel::sort(order.begin(), order.end(), [&](int64_t a, int64_t b) { return key(pairs[a]) < key(pairs[b]); });
  const int64_t np = (int64_t)pairs.size();
  out.npairs = np;
  out.pLs.resize(np); out.pLe.resize(np); out.pRs.resize(np); out.pRe.resize(np);
  out.pn.resize((size_t)nd * np); out.pJnL.resize(np); out.pJnR.resize(np);
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < np; ++i) {
    const Pair &pr = pairs[order[i]];
    out.pLs[i] = pr.Ls; out.pLe[i] = pr.Le; out.pRs[i] = pr.Rs; out.pRe[i] = pr.Re;
    for (int n = 0; n < nd; ++n) out.pn[(size_t)n * np + i] = out.fp_n[((size_t)n * Nf + pr.Ls) * ld + pr.Le];
    out.pJnL[i] = out.fp_Jn[(size_t)pr.Ls * ld + pr.Le];
    out.pJnR[i] = out.fp_Jn[(size_t)pr.Rs * ld + pr.Re];
    // element-centric tables
    out.fp_pe[(size_t)pr.Ls * ld + pr.Le] = pr.Re; out.fp_ps[(size_t)pr.Ls * ld + pr.Le] = pr.Rs;
    out.fp_pe[(size_t)pr.Rs * ld + pr.Re] = pr.Le; out.fp_ps[(size_t)pr.Rs * ld + pr.Re] = pr.Ls;
  }
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < np; ++i) {  // R side flagged by a negative J*n
    const Pair &pr = pairs[order[i]];
    out.fp_Jn[(size_t)pr.Rs * ld + pr.Re] = -out.fp_Jn[(size_t)pr.Rs * ld + pr.Re];
  }
  out.nbnd = nb * nfp;
  out.bs.resize(out.nbnd); out.be.resize(out.nbnd); out.bbc.resize(out.nbnd);
  out.bn.resize((size_t)nd * out.nbnd); out.bJn.resize(out.nbnd);
  for (int64_t b = 0; b < nb; ++b)
    for (int k = 0; k < nfp; ++k) {
      int64_t i = b * nfp + k;
      int32_t e = in.bfaces[3 * b], s = in.bfaces[3 * b + 1] * nfp + k;
      out.bs[i] = s; out.be[i] = e; out.bbc[i] = in.bfaces[3 * b + 2];
      for (int n = 0; n < nd; ++n) out.bn[(size_t)n * out.nbnd + i] = out.fp_n[((size_t)n * Nf + s) * ld + e];
      out.bJn[i] = out.fp_Jn[(size_t)s * ld + e];
      out.fp_pe[(size_t)s * ld + e] = -1 - in.bfaces[3 * b + 2]; out.fp_ps[(size_t)s * ld + e] = s;
    }
  if (!standalone) out.xf.swap(xf);
  return FR_OK;
}

}  // namespace fr
