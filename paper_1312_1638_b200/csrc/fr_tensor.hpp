// Tensor-product (sum-factorised, fused) kernels for quadrilateral / hexahedral elements.
#pragma once
#include <vector>

#include "fr_dev.hpp"
#include "fr_host.hpp"

namespace fr {

struct TensorPlan {
  int64_t work_bytes = 0;
  // workspace offsets (bytes) of the flux-point intermediates
  int64_t off_uf = 0, off_gf = 0;
  const double *ops1d = nullptr;  // device: D1, lm, lp, gm, gp, Dhat
  int variant = 0;
};

bool tensor_supported(const DevConsts &c);
cudaError_t tensor_plan(const DevConsts &c, const RefOps &o, const MeshConsts &mc, TensorPlan &tp, std::vector<void *> &allocs);
cudaError_t tensor_rhs(const DevConsts &c, const TensorPlan &tp, const void *u, void *rhs, char *work, cudaStream_t s, Prof *prof);
int tensor_rhs_launches(const DevConsts &c);

}  // namespace fr
