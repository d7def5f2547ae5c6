// Internal host-side structures of the FR library (not part of the ABI).
#pragma once
#include <cstdint>
#include <string>
#include <vector>

#include "../../include/fr.h"

namespace fr {

// Reference element + constant operator matrices (App A), built in binary128 and
// rounded once to double.  Row-major.
struct RefOps {
  int etype = 0, nd = 0, p = 0, n = 0;  // n = p+1
  int Nu = 0, Nf = 0, nfaces = 0, nfp = 0;
  std::vector<long double> xu, xf, nf;  // [Nu][nd], [Nf][nd], [Nf][nd]
  std::vector<double> wu, wf;           // quadrature weights (integral of l_rho; face GL weights)
  std::vector<double> M[7];             // M0..M6
  int64_t rows[7], cols[7];
  std::vector<double> M46;              // M4 - M6 M0   (Eq 42 :756)  [nd*Nu][Nu]
  std::vector<double> M132;             // M1 - M3 M2   (Eq 44 :773)  [Nu][nd*Nu]
  // 1-D factors of the tensor-product operators (quad/hex only)
  std::vector<double> D1;               // D1[i][j] = l_j'(xi_i)
  std::vector<double> lm, lp;           // l_j(-1), l_j(+1)
  std::vector<double> gm, gp;           // lifting coefficients: (div g) of the -1 / +1 face point at node i
  std::vector<double> Dhat;             // D1 + gm lm^T - gp lp^T   (1-D form of M1 - M3 M2; reference normal -1 on the -1 face)
  // geometry basis (degree p_g) at the solution / flux points
  int p_g = 0, Nn = 0;
  std::vector<long double> Gu, dGu, Gf, dGf;  // [Nu][Nn], [nd][Nu][Nn], [Nf][Nn], [nd][Nf][Nn]
};

void build_ref_ops(int etype, int p, int p_g, int correction, RefOps &out);  // fr_basis.cpp

// Per-mesh geometric constants and the interface lookup tables, host copies.
struct MeshConsts {
  int64_t Nel = 0, ld = 0, npairs = 0, nbnd = 0;
  std::vector<double> xu;       // [Nu][Nel][nd]
  std::vector<double> smat;     // [nd*nd][Nu][ld]   S[i][n] = J * dxi_i/dx_n     (Eq 12 :214)
  std::vector<double> rcpj;     // [Nu][ld]          1/J                           (Eq 19 :243)
  // flux-point pairs in iteration order (sorted by L flux point)
  std::vector<int32_t> pLs, pLe, pRs, pRe;  // flux point index / element of each side
  std::vector<double> pn;       // [nd][npairs] unit normal of the L side          (Eq 14 :223)
  std::vector<double> pJnL, pJnR;  // J*n of each side                             (Eq 16-17)
  // boundary flux points
  std::vector<int32_t> bs, be, bbc;
  std::vector<double> bn, bJn;  // [nd][nbnd], [nbnd]
  // per flux point (element-centric kernels): partner location, side flag, normal, J*n
  std::vector<int32_t> fp_pe, fp_ps;  // [Nf][ld] partner element / flux point (-1-bc_id at boundaries)
  std::vector<double> fp_n;     // [nd][Nf][ld] OWN outward unit normal
  std::vector<double> fp_Jn;    // [Nf][ld]; sign bit set (negative) when this flux point is the R side
  std::vector<double> xf;       // [Nf][Nel][nd] flux-point coordinates, kept only for the parts of a mixed mesh
  bool affine = false;          // every element has constant S (J) — metric arrays could be per element
};

struct MeshInput {
  int nd = 0, etype = 0, p_g = 0;
  int64_t Nel = 0;
  std::vector<double> nodes;
  std::vector<int32_t> ifaces;
  std::vector<double> shifts;
  std::vector<int32_t> bfaces;
  std::vector<fr_bc_desc> bcs;
};

// fr_mesh.cpp; returns FR_OK or an error code with text in err
// pair_block > 0: order the flux-point pairs element-block major (blocks of pair_block elements) instead of sigma major
// standalone = false (part of a mixed mesh): the part's own interface list is empty, interior flux points are left for the
// cross-part pairing of fr_api.cu (no coverage check here), and the flux-point coordinates are kept in out.xf
int build_mesh_consts(const MeshInput &in, const RefOps &ops, int64_t ld, int pair_block, MeshConsts &out, std::string &err,
                      bool standalone = true);

}  // namespace fr
