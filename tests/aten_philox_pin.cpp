// Pin helper: prints the four words of ATen's header-only Philox4x32-10 engine (a library routine,
// torch/include/ATen/core/PhiloxRNGEngine.h) for (seed, subsequence, offset) triples read from argv.
// at::Philox4_32 uses key = (seed lo, seed hi), counter = (offset lo, offset hi, subseq lo, subseq hi).
#include <ATen/core/PhiloxRNGEngine.h>
#include <cstdio>
#include <cstdlib>
int main(int argc, char** argv) {
  for (int a = 1; a + 2 < argc; a += 3) {
    const unsigned long long seed = strtoull(argv[a], 0, 0), subseq = strtoull(argv[a + 1], 0, 0),
                             off = strtoull(argv[a + 2], 0, 0);
    at::Philox4_32 e(seed, subseq, off);
    for (int i = 0; i < 4; ++i) printf("%08x ", (unsigned)e());
    printf("\n");
  }
  return 0;
}
