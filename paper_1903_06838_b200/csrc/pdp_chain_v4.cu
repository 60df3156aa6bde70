// 8-byte raw vectors (S and W multiples of 4, not of 8).
#include "pdp_chain_inst.cuh"
namespace pdp {
ChainFn chain_lookup_v4(int nv, int lps, int mode) {
  PDP_CHAIN_CASE(4, 1, 32)
  PDP_CHAIN_CASE(4, 2, 32)
  PDP_CHAIN_CASE(4, 3, 32)
  PDP_CHAIN_CASE(4, 4, 32)
  PDP_CHAIN_CASE(4, 8, 32)
  return nullptr;
}
DenseFn dense_lookup_v4(int nv, int mode) {
  PDP_DENSE_CASE(4, 1)
  PDP_DENSE_CASE(4, 2)
  PDP_DENSE_CASE(4, 4)
  PDP_DENSE_CASE(4, 8)
  return nullptr;
}
}  // namespace pdp
