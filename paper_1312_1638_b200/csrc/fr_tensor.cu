// Tensor-product kernels (placeholder until the sum-factorised hexahedral path lands).
#include "fr_tensor.hpp"

namespace fr {
bool tensor_supported(const DevConsts &) { return false; }
cudaError_t tensor_plan(const DevConsts &, const RefOps &, const MeshConsts &, TensorPlan &, std::vector<void *> &) { return cudaErrorNotSupported; }
cudaError_t tensor_rhs(const DevConsts &, const TensorPlan &, const void *, void *, char *, cudaStream_t, Prof *) { return cudaErrorNotSupported; }
int tensor_rhs_launches(const DevConsts &) { return 0; }
}  // namespace fr
