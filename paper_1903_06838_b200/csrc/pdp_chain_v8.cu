// 16-byte raw vectors (S and W multiples of 8).  (NV, LPS): vectors per lane, lanes per row segment.
#include "pdp_chain_inst.cuh"
namespace pdp {
ChainFn chain_lookup_v8(int nv, int lps, int mode) {
  PDP_CHAIN_CASE(8, 6, 8)    // S = 384 (configs[1])
  PDP_CHAIN_CASE(8, 4, 8)    // S = 256 (configs[4])
  PDP_CHAIN_CASE(8, 4, 16)   // S = 512 (configs[3])
  PDP_CHAIN_CASE(8, 3, 16)
  PDP_CHAIN_CASE(8, 2, 16)
  PDP_CHAIN_CASE(8, 1, 32)
  PDP_CHAIN_CASE(8, 2, 32)
  PDP_CHAIN_CASE(8, 3, 32)
  PDP_CHAIN_CASE(8, 4, 32)
  return nullptr;
}
DenseFn dense_lookup_v8(int nv, int mode) {
  PDP_DENSE_CASE(8, 1)
  PDP_DENSE_CASE(8, 2)
  PDP_DENSE_CASE(8, 3)
  PDP_DENSE_CASE(8, 4)
  return nullptr;
}
}  // namespace pdp
