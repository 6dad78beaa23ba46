// Test helper: exposes PyTorch's own CPU Philox4x32-10 (ATen/core/PhiloxRNGEngine.h, a
// library routine independent of oracle/ and of the CUDA path) through a C function, so
// the oracle's Philox can be pinned on the CPU.  counter = (c0,c1,c2,c3), key = (k0,k1).
#include <ATen/core/PhiloxRNGEngine.h>
#include <cstdint>
extern "C" void torch_philox4x32_10(const uint32_t* ctr, const uint32_t* key, uint32_t* out, uint64_t n) {
  for (uint64_t i = 0; i < n; ++i) {
    uint64_t seed = (uint64_t)key[2 * i] | ((uint64_t)key[2 * i + 1] << 32);
    uint64_t offs = (uint64_t)ctr[4 * i] | ((uint64_t)ctr[4 * i + 1] << 32);
    uint64_t subs = (uint64_t)ctr[4 * i + 2] | ((uint64_t)ctr[4 * i + 3] << 32);
    at::philox_engine e(seed, subs, 0);
    e.set_offset(offs);
    for (int k = 0; k < 4; ++k) out[4 * i + k] = e();
  }
}
