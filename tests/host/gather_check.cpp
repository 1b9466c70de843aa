// Host check of csrc/gather.cuh against plain bit extraction (built and run by tests/test_host_logic.py).
#include <cstdio>
#include <cstdlib>
#include "../../paper_2606_23419_b200/csrc/gather.cuh"

template <int B>
int check(unsigned seed) {
    srand(seed);
    for (int it = 0; it < 2000; ++it) {
        uint32_t W[8], V[8];
        for (int j = 0; j < 8; ++j) W[j] = ((uint32_t)rand() << 17) ^ ((uint32_t)rand() << 5) ^ (uint32_t)rand();
        gq::gather<B>(W, V);
        for (int p = 0; p < 32; ++p) {
            int code = 0;
            for (int j = 0; j < B; ++j) code |= (int)((W[j] >> p) & 1u) << (7 - j);
            int L = p >> 3, r = p & 7;
            int got = (int)((V[r] >> (8 * L)) & 0xFFu);
            if (got != code) {
                printf("FAIL B=%d p=%d code=%d got=%d\n", B, p, code, got);
                return 1;
            }
        }
    }
    return 0;
}

int main() {
    int rc = check<2>(1) | check<4>(2) | check<8>(3);
    if (!rc) printf("OK\n");
    return rc;
}
