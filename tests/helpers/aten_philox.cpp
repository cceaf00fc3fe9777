// Test helper (CPU): exposes PyTorch's own at::philox_engine (ATen/core/PhiloxRNGEngine.h, a library
// routine independent of this repository) through a C ABI, as the pin for the oracle's Philox4x32-10.
// at::philox_engine(seed, subsequence, offset): key = (seed lo, seed hi),
// counter = (offset lo, offset hi, subsequence lo, subsequence hi); operator() hands out the four
// output words of one block in order.
#include <ATen/core/PhiloxRNGEngine.h>
#include <cstdint>

extern "C" void aten_philox4x32_10(uint64_t seed, uint64_t subsequence, uint64_t offset, uint32_t out[4]) {
  at::philox_engine eng(seed, subsequence, offset);
  for (int i = 0; i < 4; ++i) out[i] = eng();
}
