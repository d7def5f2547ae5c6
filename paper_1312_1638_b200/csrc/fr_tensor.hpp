// Tensor-product (sum-factorised, fused) kernels for quadrilateral / hexahedral elements.
#pragma once
#include <vector>

#include "fr_dev.hpp"
#include "fr_host.hpp"

namespace fr {

struct TensorPlan {
  int64_t work_bytes = 0;
  // workspace offsets (bytes): U^f (-> D~), jump C - U^f, Q~ -> Q -> F~, Q^f
  int64_t off_uf = 0, off_cf = 0, off_qu = 0, off_qf = 0;
  double h_ops[2 * 64 + 4 * 8];   // host copy of the 1-D operators: D, Dhat, lm, lp, gm, gp (n <= 8)
  bool use_tma = false;           // hexahedra on the TMA-pipelined kernels (fr_hex_tma.cu); off_qu then holds G^f, off_qf the slice-major Q
};

bool tensor_supported(const DevConsts &c);
cudaError_t tensor_plan(const DevConsts &c, const RefOps &o, const MeshConsts &mc, TensorPlan &tp, std::vector<void *> &allocs);
cudaError_t tensor_rhs(const DevConsts &c, const TensorPlan &tp, const void *u, void *rhs, char *work, cudaStream_t s, Prof *prof);
int tensor_rhs_launches(const DevConsts &c);

}  // namespace fr
