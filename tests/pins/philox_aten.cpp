// Pin C1 helper: an implementation of Philox4x32-10 that is NOT ours — ATen's at::philox_engine
// (torch/include/ATen/core/PhiloxRNGEngine.h), the CPU mirror of cuRAND's Philox4_32_10 stream layout.
// at::philox_engine(seed, subsequence, offset): key = seed, counter = (offset_lo, offset_hi, subseq_lo, subseq_hi).
// Our layout (SURVEY.md §8(c) "Uniforms"): counter = (n, block, id_lo, id_hi)  <=>  offset = n + 2^32*block,
// subsequence = id.  Four successive engine outputs are the block's words w0..w3.
#include <ATen/core/PhiloxRNGEngine.h>
#include <cstdint>
extern "C" void aten_philox_block(uint64_t seed, uint64_t id, uint32_t n, uint32_t block, uint32_t out[4]) {
  at::philox_engine eng(seed, id, (uint64_t)n + ((uint64_t)block << 32));
  for (int i = 0; i < 4; ++i) out[i] = eng();
}
