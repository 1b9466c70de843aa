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

// 2-bit-segment store: X[j] byte i = left-aligned code of column 4 i + j, from NS segment words of 16 pairs each
template <int NS>
int check2(unsigned seed) {
    srand(seed);
    for (int it = 0; it < 2000; ++it) {
        uint32_t a[4], X[4];
        for (int j = 0; j < 4; ++j) a[j] = ((uint32_t)rand() << 17) ^ ((uint32_t)rand() << 5) ^ (uint32_t)rand();
        gq::gather_seg2<NS>(a, X);
        for (int c = 0; c < 16; ++c) {
            int code = 0;
            for (int sg = 0; sg < NS; ++sg) code |= (int)((a[sg] >> (2 * c)) & 3u) << (6 - 2 * sg);
            int got = (int)((X[c & 3] >> (8 * (c >> 2))) & 0xFFu);
            if (got != code) {
                printf("FAIL seg2 NS=%d c=%d code=%d got=%d\n", NS, c, code, got);
                return 1;
            }
        }
    }
    return 0;
}

int main() {
    int rc = check<2>(1) | check<4>(2) | check<8>(3) | check2<1>(4) | check2<2>(5) | check2<3>(6) | check2<4>(7);
    if (!rc) printf("OK\n");
    return rc;
}
