// Test-only helper: exposes ATen's host Philox4x32-10 engine (a library routine
// independent of both the oracle and the CUDA path) behind a C symbol.
// at::Philox4_32(seed, subsequence, offset): key = seed (lo, hi);
// counter = (offset lo, offset hi, subsequence lo, subsequence hi).
#include <ATen/core/PhiloxRNGEngine.h>
#include <cstdint>
extern "C" void aten_philox4x32_10(uint64_t seed, uint64_t subsequence, uint64_t offset, uint32_t out[4])
{
    at::Philox4_32 eng(seed, subsequence, offset);
    for (int i = 0; i < 4; ++i) out[i] = eng();
}
