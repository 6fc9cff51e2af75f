// Launch code of the Jacobian kernel for one value of LS (state pairs per item); instantiated in pyjac_jacobian_ls*.cu
// (one translation unit per LS so that they compile in parallel).
#pragma once
#include "pyjac_jacobian.cuh"

namespace pyjac {

template <int LS> int jac2_set_attr() {
  cudaError_t e = cudaFuncSetAttribute(jac2::jacobian2_kernel<LS, false, uint16_t>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)J_SMEM_LIMIT);
  if (e != cudaSuccess) return (int)e;
  e = cudaFuncSetAttribute(jac2::jacobian2_kernel<LS, false, uint32_t>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)J_SMEM_LIMIT);
  if (e != cudaSuccess) return (int)e;
  return (int)cudaFuncSetAttribute(jac2::jacobian2_kernel<LS, true, uint32_t>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)J_SMEM_LIMIT);
}

template <int LS> int jac2_launch(const DevJac& m, const DevJacOut& o, size_t smem, int n_sm, int mode, int64_t n_states, int64_t tile,
                                  const double* phi, const double* param, double* out, unsigned long long* sched, cudaStream_t st) {
  const int64_t tiles = (n_states + 2 * LS - 1) / (2 * LS);
  if (tiles == 0) return 0;
  const unsigned blocks = (unsigned)std::min<int64_t>(tiles, (int64_t)n_sm);   // persistent: one CTA per SM
  int tshift = -1;                                  // log2(tile) if tile is a power of two, else tile == ld
  if ((tile & (tile - 1)) == 0) { tshift = 0; while (((int64_t)1 << tshift) < tile) ++tshift; }
  if (o.nzmask != nullptr) jac2::jacobian2_kernel<LS, true, uint32_t><<<blocks, J_NT, smem, st>>>(m, o, mode, n_states, tile, tshift, phi, param, out, sched);
  else if (o.pos16) jac2::jacobian2_kernel<LS, false, uint16_t><<<blocks, J_NT, smem, st>>>(m, o, mode, n_states, tile, tshift, phi, param, out, sched);
  else jac2::jacobian2_kernel<LS, false, uint32_t><<<blocks, J_NT, smem, st>>>(m, o, mode, n_states, tile, tshift, phi, param, out, sched);
  return (int)cudaGetLastError();
}

}  // namespace pyjac
