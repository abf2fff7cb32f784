// dmx_inst.cuh — launcher definitions; each inst_*.cu instantiates them for one (real type, lanes)
// pair so that the translation units compile in parallel.
#pragma once
#include "dmx_adjoint.cuh"

namespace dmx {

template <class R, int G, class SH> cudaError_t launch_rollout(const ModelDev<R>& m, const RolloutArgs<R>& a, LaunchCfg c, cudaStream_t s) {
  cudaError_t e = cudaFuncSetAttribute(rollout_kernel<R, G, SH>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c.smem);
  if (e != cudaSuccess) return e;
  rollout_kernel<R, G, SH><<<c.grid, c.block, c.smem, s>>>(m, a);
  return cudaGetLastError();
}
template <class R, int G, class SH> cudaError_t launch_backward(const ModelDev<R>& m, const BackwardArgs<R>& a, LaunchCfg c, cudaStream_t s) {
  cudaError_t e = cudaFuncSetAttribute(backward_kernel<R, G, SH>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c.smem);
  if (e != cudaSuccess) return e;
  backward_kernel<R, G, SH><<<c.grid, c.block, c.smem, s>>>(m, a);
  return cudaGetLastError();
}
template <class R, int G, class SH> cudaError_t launch_backward_ckpt(const ModelDev<R>& m, const BackwardArgs<R>& a, LaunchCfg c, cudaStream_t s) {
  cudaError_t e = cudaFuncSetAttribute(backward_kernel<R, G, SH, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c.smem);
  if (e != cudaSuccess) return e;
  backward_kernel<R, G, SH, true><<<c.grid, c.block, c.smem, s>>>(m, a);
  return cudaGetLastError();
}
template <class R, int G, class SH> cudaError_t launch_adjoint(const ModelDev<R>& m, const AdjointArgs<R>& a, LaunchCfg c, cudaStream_t s) {
  cudaError_t e = cudaFuncSetAttribute(adjoint_kernel<R, G, SH>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c.smem);
  if (e != cudaSuccess) return e;
  adjoint_kernel<R, G, SH><<<c.grid, c.block, c.smem, s>>>(m, a);
  return cudaGetLastError();
}
template <class R, int G, class SH> cudaError_t launch_field(const ModelDev<R>& m, const FieldArgs<R>& a, LaunchCfg c, cudaStream_t s) {
  cudaError_t e = cudaFuncSetAttribute(field_kernel<R, G, SH>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c.smem);
  if (e != cudaSuccess) return e;
  field_kernel<R, G, SH><<<c.grid, c.block, c.smem, s>>>(m, a);
  return cudaGetLastError();
}
template <class R, int G, class SH> cudaError_t launch_invweight(const ModelDev<R>& m, const R* qpos0, const R* zero_v, R* body_w, const WsLayout& wl,
                                                       const RkLayout& rl, LaunchCfg c, cudaStream_t s) {
  cudaError_t e = cudaFuncSetAttribute(invweight_kernel<R, G, SH>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c.smem);
  if (e != cudaSuccess) return e;
  invweight_kernel<R, G, SH><<<1, c.block, c.smem, s>>>(m, qpos0, zero_v, body_w, wl, rl);
  return cudaGetLastError();
}
template <class R, int G, class SH> cudaError_t launch_prof_dump(unsigned long long* out, cudaStream_t s) {
  prof_dump_kernel<R, G, SH><<<1, 32, 0, s>>>(out);
  return cudaGetLastError();
}
template <class R, int G, class SH> cudaError_t kernel_occupancy(int block, size_t smem_fwd, size_t smem_bwd, size_t smem_field, int* occ_fwd, int* occ_bwd, int* occ_field) {
  cudaError_t e = cudaFuncSetAttribute(rollout_kernel<R, G, SH>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_fwd);
  if (e != cudaSuccess) return e;
  e = cudaFuncSetAttribute(backward_kernel<R, G, SH>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bwd);
  if (e != cudaSuccess) return e;
  e = cudaFuncSetAttribute(field_kernel<R, G, SH>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_field);
  if (e != cudaSuccess) return e;
  e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(occ_fwd, rollout_kernel<R, G, SH>, block, smem_fwd);
  if (e != cudaSuccess) return e;
  e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(occ_bwd, backward_kernel<R, G, SH>, block, smem_bwd);
  if (e != cudaSuccess) return e;
  return cudaOccupancyMaxActiveBlocksPerMultiprocessor(occ_field, field_kernel<R, G, SH>, block, smem_field);
}

}  // namespace dmx

#define DMX_INSTANTIATE(R, G, SH)                                                                                                  \
  template cudaError_t dmx::launch_rollout<R, G, dmx::SH>(const dmx::ModelDev<R>&, const dmx::RolloutArgs<R>&, dmx::LaunchCfg, cudaStream_t);   \
  template cudaError_t dmx::launch_backward<R, G, dmx::SH>(const dmx::ModelDev<R>&, const dmx::BackwardArgs<R>&, dmx::LaunchCfg, cudaStream_t); \
  template cudaError_t dmx::launch_backward_ckpt<R, G, dmx::SH>(const dmx::ModelDev<R>&, const dmx::BackwardArgs<R>&, dmx::LaunchCfg, cudaStream_t); \
  template cudaError_t dmx::launch_adjoint<R, G, dmx::SH>(const dmx::ModelDev<R>&, const dmx::AdjointArgs<R>&, dmx::LaunchCfg, cudaStream_t); \
  template cudaError_t dmx::launch_field<R, G, dmx::SH>(const dmx::ModelDev<R>&, const dmx::FieldArgs<R>&, dmx::LaunchCfg, cudaStream_t);       \
  template cudaError_t dmx::launch_invweight<R, G, dmx::SH>(const dmx::ModelDev<R>&, const R*, const R*, R*, const dmx::WsLayout&,             \
                                                            const dmx::RkLayout&, dmx::LaunchCfg, cudaStream_t);                             \
  template cudaError_t dmx::launch_prof_dump<R, G, dmx::SH>(unsigned long long*, cudaStream_t);                                              \
  template cudaError_t dmx::kernel_occupancy<R, G, dmx::SH>(int, size_t, size_t, size_t, int*, int*, int*);
