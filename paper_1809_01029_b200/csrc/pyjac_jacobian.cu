// Dispatch of the analytical Jacobian kernel (pyjac_jacobian.cuh) over LS, the number of state pairs per item.
#include <cuda_runtime.h>

#include <algorithm>

#include "pyjac_internal.h"

namespace pyjac {

template <int LS> int jac2_set_attr();
template <int LS> int jac2_launch(const DevJac&, const DevJacOut&, size_t, int, int, int64_t, int64_t, const double*, const double*, double*,
                                  unsigned long long*, cudaStream_t);

// The largest tile (2 LS states) whose intermediates fit in shared memory and that still leaves two tiles per SM:
// more states per CTA amortise the plan and table reads (L2 -> SM traffic per state falls with LS).
LaunchCfg choose_cfg_jac(const JacTables& j, int64_t tile, int64_t n_states, int n_sm) {
  (void)tile;          // any layout works with any LS: a thread addresses its two states individually
  LaunchCfg cfg{2, J_NT, jac_smem_bytes(j, 1)};
  for (int LS = 4; LS >= 1; LS >>= 1) {
    const size_t bytes = jac_smem_bytes(j, LS);
    if (bytes > J_SMEM_LIMIT && LS > 1) continue;
    if (LS > 1 && (n_states + 2 * LS - 1) / (2 * LS) < 2 * (int64_t)n_sm) continue;
    cfg.S = 2 * LS; cfg.smem = bytes;
    break;
  }
  return cfg;
}

int launch_jacobian2(const DevJac& m, const DevJacOut& o, const LaunchCfg& cfg, int n_sm, int mode, int64_t n_states, int64_t tile,
                     const double* phi, const double* param, double* out, unsigned long long* sched, void* stream) {
  cudaStream_t st = (cudaStream_t)stream;
  switch (cfg.S) {
    case 8: return jac2_launch<4>(m, o, cfg.smem, n_sm, mode, n_states, tile, phi, param, out, sched, st);
    case 4: return jac2_launch<2>(m, o, cfg.smem, n_sm, mode, n_states, tile, phi, param, out, sched, st);
    default: return jac2_launch<1>(m, o, cfg.smem, n_sm, mode, n_states, tile, phi, param, out, sched, st);
  }
}

int set_kernel_attributes_jac() {
  int e;
  if ((e = jac2_set_attr<1>())) return e;
  if ((e = jac2_set_attr<2>())) return e;
  return jac2_set_attr<4>();
}

}  // namespace pyjac
