// Jacobian kernel, 2 states per CTA (LS = 1 state pairs per item)
#include <algorithm>

#include "pyjac_jacobian_launch.cuh"

namespace pyjac {
template int jac2_set_attr<1>();
template int jac2_launch<1>(const DevJac&, const DevJacOut&, size_t, int, int, int64_t, int64_t, const double*, const double*, double*,
                             unsigned long long*, cudaStream_t);
}  // namespace pyjac

