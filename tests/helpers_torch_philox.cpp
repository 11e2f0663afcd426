// Test helper: prints raw outputs of PyTorch's header-only at::philox_engine
// (ATen/core/PhiloxRNGEngine.h), an implementation of Philox4x32-10 independent of
// oracle/ and of the CUDA path.  Usage: helper seed subsequence offset n
#include <ATen/core/PhiloxRNGEngine.h>
#include <cstdio>
#include <cstdlib>
int main(int argc, char** argv) {
    if (argc < 5) return 2;
    const uint64_t seed = strtoull(argv[1], nullptr, 0);
    const uint64_t subsequence = strtoull(argv[2], nullptr, 0);
    const uint64_t offset = strtoull(argv[3], nullptr, 0);
    const int n = atoi(argv[4]);
    at::philox_engine eng(seed, subsequence, offset);
    for (int i = 0; i < n; ++i) printf("%u\n", (unsigned)eng());
    return 0;
}
