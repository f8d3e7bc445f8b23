// Test helper: prints Philox4x32-10 outputs from torch's own at::philox_engine
// (ATen/core/PhiloxRNGEngine.h), an implementation independent of oracle/ and of the CUDA path.
// stdin: lines "c0 c1 c2 c3 k0 k1" (decimal); stdout: "o0 o1 o2 o3" per line.
#include <ATen/core/PhiloxRNGEngine.h>
#include <cstdint>
#include <cstdio>

int main() {
  unsigned long long c0, c1, c2, c3, k0, k1;
  while (std::scanf("%llu %llu %llu %llu %llu %llu", &c0, &c1, &c2, &c3, &k0, &k1) == 6) {
    const uint64_t seed = (uint64_t)k0 | ((uint64_t)k1 << 32);
    const uint64_t subsequence = (uint64_t)c2 | ((uint64_t)c3 << 32);
    const uint64_t offset = (uint64_t)c0 | ((uint64_t)c1 << 32);
    at::philox_engine e(seed, subsequence, offset);
    const uint32_t o0 = e(), o1 = e(), o2 = e(), o3 = e();
    std::printf("%u %u %u %u\n", o0, o1, o2, o3);
  }
  return 0;
}
