// Independent Philox4x32-10 for pinning the oracle's generator: PyTorch's header-only at::Philox4_32
// (ATen/core/PhiloxRNGEngine.h, shipped with the torch wheel).  counter = (offset_lo, offset_hi, subseq_lo,
// subseq_hi), key = (seed_lo, seed_hi); operator() returns the four words of one block in order.
// Usage: philox_aten_ref < lines of "c0 c1 c2 c3 k0 k1" (hex)  ->  lines of "w0 w1 w2 w3" (hex)
#include <ATen/core/PhiloxRNGEngine.h>
#include <cstdio>
#include <cstdint>
int main() {
  unsigned c0, c1, c2, c3, k0, k1;
  while (scanf("%x %x %x %x %x %x", &c0, &c1, &c2, &c3, &k0, &k1) == 6) {
    at::Philox4_32 e((uint64_t)k0 | ((uint64_t)k1 << 32), (uint64_t)c2 | ((uint64_t)c3 << 32), (uint64_t)c0 | ((uint64_t)c1 << 32));
    unsigned w0 = e(), w1 = e(), w2 = e(), w3 = e();
    printf("%08x %08x %08x %08x\n", w0, w1, w2, w3);
  }
  return 0;
}
