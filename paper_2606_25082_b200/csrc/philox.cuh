// philox.cuh -- the ONE Philox4x32-10 of libmigsim.so (R1), used by the rollout kernels, the arrival generator
// and the Q-network's epsilon-greedy policy.  Nothing here is shared with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace migsim {

// Salmon, Moraes, Dror, Shaw (SC'11): ten rounds of two 32x32->64 multiplies; the key is bumped by the Weyl constants
// between rounds.  counter (c0..c3) = (index, stream, global env id, episode), key (k0, k1) = the seed's halves.
__device__ __forceinline__ uint4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0, uint32_t k1) {
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
    uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
    uint32_t n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
    c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
    k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
  }
  return make_uint4(c0, c1, c2, c3);
}

}  // namespace migsim
