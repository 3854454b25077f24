// Test helper (host-only build): prints cuRAND's own Philox4x32-10 block function,
// taken from the CUDA toolkit header, for counters/keys given on the command line.
// Used to pin the oracle's Philox (tests/test_oracle_rng.py).  Not part of the product.
#define QUALIFIERS static inline __host__ __device__
#include <cstdio>
#include <cstdlib>
#include <curand_philox4x32_x.h>
int main(int argc, char** argv)
{
    for (int i = 1; i + 5 < argc; i += 6) {
        uint4 c = make_uint4(strtoul(argv[i], 0, 10), strtoul(argv[i + 1], 0, 10), strtoul(argv[i + 2], 0, 10), strtoul(argv[i + 3], 0, 10));
        uint2 k = make_uint2(strtoul(argv[i + 4], 0, 10), strtoul(argv[i + 5], 0, 10));
        uint4 r = curand_Philox4x32_10(c, k);
        printf("%u %u %u %u\n", r.x, r.y, r.z, r.w);
    }
    return 0;
}
