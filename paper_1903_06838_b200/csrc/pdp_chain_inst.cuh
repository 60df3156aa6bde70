// pdp_chain_inst.cuh — explicit instantiation tables of pdp_chain_kernel<V, NV, LPS, MODE>, one translation unit
// per vector width so that the variants compile in parallel (pdp_chain_v8.cu, pdp_chain_v4.cu, pdp_chain_v2.cu).
#pragma once
#include "pdp_chain.cuh"
#include "pdp_dense.cuh"

namespace pdp {
using ChainFn = void (*)(const CParams);

template <int V, int NV, int LPS>
inline ChainFn chain_modes(int mode) {
  return mode == 0 ? pdp_chain_kernel<V, NV, LPS, 0> : (mode == 1 ? pdp_chain_kernel<V, NV, LPS, 1> : pdp_chain_kernel<V, NV, LPS, 2>);
}
}  // namespace pdp

namespace pdp {
using DenseFn = void (*)(const DParams);
template <int V, int NV>
inline DenseFn dense_modes(int mode) {
  return mode == 0 ? pdp_dense_kernel<V, NV, 0> : (mode == 1 ? pdp_dense_kernel<V, NV, 1> : pdp_dense_kernel<V, NV, 2>);
}
}  // namespace pdp
#define PDP_DENSE_CASE(V, NV) \
  if (nv == NV) return pdp::dense_modes<V, NV>(mode);

#define PDP_CHAIN_CASE(V, NV, LPS) \
  if (nv == NV && lps == LPS) return pdp::chain_modes<V, NV, LPS>(mode);
