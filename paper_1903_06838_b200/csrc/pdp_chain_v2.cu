// 4-byte raw vectors (any even S and W; configs[0], configs[2]: S = 194).
#include "pdp_chain_inst.cuh"
namespace pdp {
ChainFn chain_lookup_v2(int nv, int lps, int mode) {
  PDP_CHAIN_CASE(2, 13, 8)   // S = 194
  PDP_CHAIN_CASE(2, 7, 16)
  PDP_CHAIN_CASE(2, 1, 32)
  PDP_CHAIN_CASE(2, 2, 32)
  PDP_CHAIN_CASE(2, 4, 32)
  PDP_CHAIN_CASE(2, 8, 32)
  PDP_CHAIN_CASE(2, 16, 32)
  return nullptr;
}
DenseFn dense_lookup_v2(int nv, int mode) {
  PDP_DENSE_CASE(2, 1)
  PDP_DENSE_CASE(2, 2)
  PDP_DENSE_CASE(2, 4)
  PDP_DENSE_CASE(2, 8)
  PDP_DENSE_CASE(2, 16)
  return nullptr;
}
}  // namespace pdp
