// grinqh_oracle.cpp — TEST INFRASTRUCTURE ONLY.
//
// Plain, slow, single-threaded CPU oracle for the GRINQH decode hot path
// (arxiv/paper_2606_23419; citations are PAPER.md:LINE).  It defines what the
// CUDA library must compute.  Only tests/, __graft_entry__.smoke() and
// bench.py's cpu_baseline / --impl reference leg may load it.  It shares no
// code, header, table or helper with paper_2606_23419_b200/csrc/.
//
// Arithmetic: integer work is exact; every floating-point accumulation is
// fp64.  The quantiser's fp32 steps are the ones DESIGN.md reading #8 fixes
// (IEEE fp32 subtract / divide, round-half-even) so that codes are bit-exact;
// build with -O2 -ffp-contract=off, never -ffast-math.
//
// Parity pins: tests/test_oracle_*.py (closed forms, invariants, brute force,
// numpy float16 / float64 library routines).  The quantiser's rounding and
// fp16-scale conventions (reading #8) are this build's: "parity unpinned"
// against the authors' unpublished code, pinned by the properties the paper
// states (nested codes PAPER.md:79, reconstruction PAPER.md:85).
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <numeric>
#include <vector>

namespace {

// ---------------------------------------------------------------- fp16 <-> fp32
// Own bit-level conversions (no _Float16, no CUDA headers).
float half_to_float(uint16_t h) {
    uint32_t sign = (uint32_t)(h & 0x8000u) << 16;
    uint32_t exp = (h >> 10) & 0x1Fu;
    uint32_t man = h & 0x3FFu;
    uint32_t out;
    if (exp == 0) {
        if (man == 0) {
            out = sign;
        } else {  // subnormal: normalise
            int e = -1;
            do {
                man <<= 1;
                ++e;
            } while ((man & 0x400u) == 0);
            man &= 0x3FFu;
            out = sign | ((uint32_t)(127 - 15 - e) << 23) | (man << 13);
        }
    } else if (exp == 31) {
        out = sign | 0x7F800000u | (man << 13);
    } else {
        out = sign | ((exp + 127 - 15) << 23) | (man << 13);
    }
    float f;
    std::memcpy(&f, &out, 4);
    return f;
}

uint16_t float_to_half(float f) {  // round to nearest even
    uint32_t x;
    std::memcpy(&x, &f, 4);
    uint16_t sign = (uint16_t)((x >> 16) & 0x8000u);
    uint32_t absx = x & 0x7FFFFFFFu;
    if (absx >= 0x7F800000u) {  // inf / nan
        if (absx == 0x7F800000u) return sign | 0x7C00u;
        return sign | 0x7C00u | 0x200u | (uint16_t)((absx >> 13) & 0x3FFu);
    }
    if (absx >= 0x477FF000u) return sign | 0x7C00u;  // >= 65520 rounds to inf
    if (absx < 0x33000001u) return sign;             // <= 2^-25 rounds to zero (tie -> even = 0)
    int32_t e = (int32_t)(absx >> 23) - 127;
    uint32_t m = (absx & 0x7FFFFFu) | 0x800000u;  // 24-bit significand
    int shift;
    uint32_t base;
    if (e < -14) {  // subnormal half
        shift = 13 + (-14 - e);
        base = 0;
    } else {
        shift = 13;
        base = (uint32_t)(e + 15) << 10;
        m &= 0x7FFFFFu;
    }
    uint32_t q = m >> shift;
    uint32_t rem = m & ((1u << shift) - 1u);
    uint32_t halfway = 1u << (shift - 1);
    uint32_t r = base + q;  // carry from mantissa into exponent is the correct rounding
    if (rem > halfway || (rem == halfway && (r & 1u))) r += 1;
    return sign | (uint16_t)r;
}

inline int phi_of(int b) {  // midpoint bias, PAPER.md:85 (phi = 2^(bmax-b-1)); reading #5: phi_8 = 0
    return (b >= 1 && b <= 7) ? (1 << (7 - b)) : 0;
}

// truncated code with midpoint bit: (q_b << (8-b)) | phi_b
inline int code_prime(int q, int b) {
    if (b <= 0) return 0;
    int mask = (0xFF << (8 - b)) & 0xFF;
    return (q & mask) | phi_of(b);
}

// re-assemble the code of (k, n) from the first `b` planes only (nested property)
inline int code_from_planes(const uint32_t* planes, int K, int N, int k, int n, int b) {
    const size_t words = (size_t)N / 32;
    const size_t plane_stride = (size_t)K * words;
    int q = 0;
    for (int j = 0; j < b; ++j) {
        uint32_t w = planes[(size_t)j * plane_stride + (size_t)k * words + (size_t)(n >> 5)];
        q |= (int)((w >> (n & 31)) & 1u) << (7 - j);
    }
    return q;
}


// ---- the paper's own granularity — 2-bit significance segments, b in {0, 2, .., bmax},
//      bmax in {4, 6, 8} (PAPER.md:79-81 "decomposed into discrete 2-bit segments", :95, :262, :440-444).
// Layout of this build, defined here by formula (reading #10b): segs[sigma][k][n >> 4], sigma = 0 is the most
// significant pair; column n's pair sits at bits 2 (n & 15) + 1 (code bit bmax - 1 - 2 sigma) and 2 (n & 15)
// (code bit bmax - 2 - 2 sigma) of the word: sixteen 2-bit chunks per uint32.
inline int phi2_of(int b, int bmax) {  // phi = 2^(bmax - b - 1); reading #5: 0 at b = bmax
    return (b >= 1 && b < bmax) ? (1 << (bmax - b - 1)) : 0;
}
inline int code2_prime(int q, int b, int bmax) {  // q_b 2^(bmax - b) + phi, q_b = the top b bits of the bmax-bit code
    if (b <= 0) return 0;
    int qb = q >> (bmax - b);
    return (qb << (bmax - b)) | phi2_of(b, bmax);
}
inline int code_from_segs(const uint32_t* segs, int K, int N, int k, int n, int b, int bmax) {
    const size_t words = (size_t)N / 16;
    const size_t seg_stride = (size_t)K * words;
    int q = 0;
    for (int sg = 0; sg < b / 2; ++sg) {  // only the first b / 2 segments are read (nested property)
        uint32_t w = segs[(size_t)sg * seg_stride + (size_t)k * words + (size_t)(n >> 4)];
        q |= (int)((w >> (2 * (n & 15))) & 3u) << (bmax - 2 - 2 * sg);
    }
    return q;
}

}  // namespace

extern "C" {

float orc_half_to_float(uint16_t h) { return half_to_float(h); }
uint16_t orc_float_to_half(float f) { return float_to_half(f); }
int orc_code_prime(int q, int b) { return code_prime(q, b); }

// DESIGN.md reading #3: fractions -> integer row counts, cumulative rounding from the top width.
int orc_mix_to_counts(int K, const double* frac, uint32_t* counts) {
    double sum = 0;
    for (int w = 0; w < 9; ++w) {
        if (!(frac[w] >= 0)) return -4;
        sum += frac[w];
    }
    if (std::fabs(sum - 1.0) > 1e-6) return -4;
    long long C[10];
    C[9] = 0;
    double F = 0;
    for (int w = 8; w >= 1; --w) {
        F += frac[w];
        long long c = (long long)std::floor(F * (double)K + 0.5);
        c = std::min<long long>(std::max<long long>(c, C[w + 1]), K);
        C[w] = c;
    }
    C[0] = K;
    for (int w = 0; w < 9; ++w) counts[w] = (uint32_t)(C[w] - C[w + 1]);
    return 0;
}

// c.1 — 8-bit asymmetric min/max RTN per (group of G rows, column), split into 8 bit planes.
// PAPER.md:79 (nested codes), :83 (s and z at full b_max precision), :95 (RTN, G = 128).
int orc_pack(const uint16_t* W, int K, int N, int G, uint32_t* planes, uint16_t* scales, uint16_t* zeros) {
    if (K % G || N % 32) return -2;
    const size_t words = (size_t)N / 32;
    const size_t plane_stride = (size_t)K * words;
    std::memset(planes, 0, sizeof(uint32_t) * 8 * plane_stride);
    for (int g = 0; g < K / G; ++g) {
        for (int n = 0; n < N; ++n) {
            // 1. exact min / max of the group's fp16 values
            float lo = half_to_float(W[(size_t)(g * G) * N + n]);
            float hi = lo;
            uint16_t lo_bits = W[(size_t)(g * G) * N + n];
            for (int i = 1; i < G; ++i) {
                uint16_t hb = W[(size_t)(g * G + i) * N + n];
                float v = half_to_float(hb);
                if (v < lo) {
                    lo = v;
                    lo_bits = hb;
                }
                if (v > hi) hi = v;
            }
            // a group whose minimum is -0.0 / +0.0: store z = +0.0 or the pattern met first; the
            // value is what matters.  Canonicalise zero to +0.0 so both sides agree bit-exactly.
            if (lo == 0.0f) lo_bits = 0;
            // 2. scale and zero
            volatile float range = hi - lo;      // IEEE fp32 subtract
            volatile float s32 = range / 255.0f;  // IEEE fp32 divide
            uint16_t s_bits = float_to_half(s32);
            float s = half_to_float(s_bits);
            float z = half_to_float(lo_bits);
            scales[(size_t)g * N + n] = s_bits;
            zeros[(size_t)g * N + n] = lo_bits;
            // 3. codes against the STORED fp16 scale
            for (int i = 0; i < G; ++i) {
                int k = g * G + i;
                int q = 0;
                if (s != 0.0f) {
                    volatile float d = half_to_float(W[(size_t)k * N + n]) - z;
                    volatile float t = d / s;
                    float r = std::nearbyintf(t);  // round-half-even in the default rounding mode
                    if (r < 0.0f) r = 0.0f;
                    if (r > 255.0f) r = 255.0f;
                    q = (int)r;
                }
                // 4. bit planes: plane j holds code bit (7 - j); column n at bit (n & 31)
                for (int j = 0; j < 8; ++j) {
                    if ((q >> (7 - j)) & 1)
                        planes[(size_t)j * plane_stride + (size_t)k * words + (size_t)(n >> 5)] |= 1u << (n & 31);
                }
            }
        }
    }
    return 0;
}

// full 8-bit codes back out of the planes (test helper)
int orc_codes(const uint32_t* planes, int K, int N, uint8_t* q) {
    for (int k = 0; k < K; ++k)
        for (int n = 0; n < N; ++n) q[(size_t)k * N + n] = (uint8_t)code_from_planes(planes, K, N, k, n, 8);
    return 0;
}

// definitional rank: r_k = #{j : m_j > m_k} + #{j < k : m_j = m_k}, O(K^2)
int orc_rank_bruteforce(const uint16_t* x, int K, int32_t* rank) {
    for (int k = 0; k < K; ++k) {
        int mk = x[k] & 0x7FFF, r = 0;
        for (int j = 0; j < K; ++j) {
            int mj = x[j] & 0x7FFF;
            if (mj > mk || (mj == mk && j < k)) ++r;
        }
        rank[k] = r;
    }
    return 0;
}

// union over tokens and the compacted lists from per-token widths (shared by the rank and threshold forms)
static void lists_from_bits(const uint8_t* bits, int T, int K, int G, uint8_t* bits_union, int32_t* rows,
                            int32_t* cnt_ge, uint8_t* grows, uint8_t* gcnt_ge, int gcnt_stride) {
    std::vector<int32_t> order(K);
    for (int k = 0; k < K; ++k) {
        uint8_t m = 0;
        for (int t = 0; t < T; ++t) m = std::max(m, bits[(size_t)t * K + k]);
        bits_union[k] = m;
    }
    // rows: (bits_union desc, k asc)
    std::iota(order.begin(), order.end(), 0);
    std::stable_sort(order.begin(), order.end(), [&](int32_t a, int32_t b) { return bits_union[a] > bits_union[b]; });
    for (int i = 0; i < K; ++i) rows[i] = order[i];
    for (int w = 0; w < 10; ++w) {
        int c = 0;
        for (int k = 0; k < K; ++k) c += (bits_union[k] >= w);
        cnt_ge[w] = c;
    }
    // per-group lists
    std::vector<int> loc(G);
    for (int g = 0; g < K / G; ++g) {
        std::iota(loc.begin(), loc.end(), 0);
        std::stable_sort(loc.begin(), loc.end(),
                         [&](int a, int b) { return bits_union[g * G + a] > bits_union[g * G + b]; });
        for (int i = 0; i < G; ++i) grows[(size_t)g * G + i] = (uint8_t)loc[i];
        for (int w = 0; w < gcnt_stride; ++w) {
            int c = 0;
            if (w < 10)
                for (int i = 0; i < G; ++i) c += (bits_union[g * G + i] >= w);
            gcnt_ge[(size_t)g * gcnt_stride + w] = (uint8_t)c;
        }
    }
}


// c.2 — rank / top-p assignment (PAPER.md:61-65 with the per-vector top-p partition of :271).
int orc_assign(const uint16_t* x, int T, int K, int G, const uint32_t* counts, uint8_t* bits, uint8_t* bits_union,
               int32_t* rows, int32_t* cnt_ge, uint8_t* grows, uint8_t* gcnt_ge, int gcnt_stride) {
    if (K % G || G > 256) return -2;
    unsigned long long total = 0;
    for (int w = 0; w < 9; ++w) total += counts[w];
    if (total != (unsigned long long)K) return -4;
    long long C[10];
    C[9] = 0;
    for (int w = 8; w >= 0; --w) C[w] = C[w + 1] + counts[w];
    std::vector<int32_t> order(K);
    for (int t = 0; t < T; ++t) {
        const uint16_t* xt = x + (size_t)t * K;
        std::iota(order.begin(), order.end(), 0);
        std::stable_sort(order.begin(), order.end(),
                         [&](int32_t a, int32_t b) { return (xt[a] & 0x7FFF) > (xt[b] & 0x7FFF); });
        for (int r = 0; r < K; ++r) {
            int b = 0;
            for (int w = 8; w >= 1; --w)
                if (r < C[w]) {
                    b = w;
                    break;
                }
            bits[(size_t)t * K + order[r]] = (uint8_t)b;
        }
    }
    lists_from_bits(bits, T, K, G, bits_union, rows, cnt_ge, grows, gcnt_ge, gcnt_stride);
    return 0;
}

// f1 — threshold assignment, the paper's run-time form (b_i = b_k if |x_i| in [theta_k, theta_{k+1})).
// theta[w], w = 1..8: the smallest fp16 magnitude pattern that still gets at least w bits, non-decreasing in w;
// 0x8000 (above every magnitude) = width w is unreachable.  theta[0] is ignored.  b = max{w : m >= theta[w]}.
int orc_assign_thresholds(const uint16_t* x, int T, int K, int G, const uint16_t* theta, uint8_t* bits,
                          uint8_t* bits_union, int32_t* rows, int32_t* cnt_ge, uint8_t* grows, uint8_t* gcnt_ge,
                          int gcnt_stride) {
    if (K % G || G > 256) return -2;
    for (int w = 2; w <= 8; ++w)
        if (theta[w] < theta[w - 1] || theta[w] > 0x8000) return -4;
    for (int t = 0; t < T; ++t)
        for (int k = 0; k < K; ++k) {
            const int m = x[(size_t)t * K + k] & 0x7FFF;
            int b = 0;
            for (int w = 1; w <= 8; ++w)
                if (m >= (int)theta[w]) b = w;
            bits[(size_t)t * K + k] = (uint8_t)b;
        }
    lists_from_bits(bits, T, K, G, bits_union, rows, cnt_ge, grows, gcnt_ge, gcnt_stride);
    return 0;
}

// Calibration of the thresholds (Eq. 2): for every calibration vector the magnitude that
// separates the levels under the rank partition (the C_w-th largest |x|, i.e. the smallest one that still gets
// >= w bits), averaged over the S vectors in fp64, rounded to fp32 and then to fp16 (both round-to-nearest-even).
// C_w == 0 -> 0x8000 (unreachable).
int orc_calibrate_thresholds(const uint16_t* xs, int S, int K, const uint32_t* counts, uint16_t* theta) {
    unsigned long long total = 0;
    for (int w = 0; w < 9; ++w) total += counts[w];
    if (total != (unsigned long long)K || S < 1) return -4;
    long long C[10];
    C[9] = 0;
    for (int w = 8; w >= 0; --w) C[w] = C[w + 1] + counts[w];
    std::vector<int> mags(K);
    double sum[9] = {0, 0, 0, 0, 0, 0, 0, 0, 0};
    for (int s = 0; s < S; ++s) {
        for (int k = 0; k < K; ++k) mags[k] = xs[(size_t)s * K + k] & 0x7FFF;
        std::sort(mags.begin(), mags.end(), [](int a, int b) { return a > b; });
        for (int w = 1; w <= 8; ++w)
            if (C[w] > 0) sum[w] += (double)half_to_float((uint16_t)mags[C[w] - 1]);
    }
    theta[0] = 0;
    for (int w = 1; w <= 8; ++w) theta[w] = (C[w] > 0) ? float_to_half((float)(sum[w] / S)) : (uint16_t)0x8000;
    return 0;
}

// c.3 — definition: y[t][n] = sum_{k : b_tk > 0} x_tk * ( s * code'(q_kn, b_tk) + z ), fp64.
// `cols` (optional): compute only those output columns, y is then [T][ncols].
int orc_vmm_cols(const uint16_t* x, int T, int K, int N, int G, const uint32_t* planes, const uint16_t* scales,
                 const uint16_t* zeros, const uint8_t* bits, const int32_t* cols, int ncols, double* y) {
    for (int t = 0; t < T; ++t) {
        for (int c = 0; c < ncols; ++c) {
            int n = cols ? cols[c] : c;
            double acc = 0.0;
            for (int k = 0; k < K; ++k) {
                int b = bits[(size_t)t * K + k];
                if (b == 0) continue;  // reading #7: bypassed channel contributes exactly 0
                int g = k / G;
                int q = code_from_planes(planes, K, N, k, n, b);  // only planes j < b are read
                double s = (double)half_to_float(scales[(size_t)g * N + n]);
                double z = (double)half_to_float(zeros[(size_t)g * N + n]);
                double what = s * (double)code_prime(q, b) + z;
                acc += (double)half_to_float(x[(size_t)t * K + k]) * what;
            }
            y[(size_t)t * ncols + c] = acc;
        }
    }
    return 0;
}

int orc_vmm(const uint16_t* x, int T, int K, int N, int G, const uint32_t* planes, const uint16_t* scales,
            const uint16_t* zeros, const uint8_t* bits, double* y) {
    return orc_vmm_cols(x, T, K, N, G, planes, scales, zeros, bits, nullptr, N, y);
}

// Second, independently written formulation: plane-wise masked accumulation.
//   sum_k x_k trunc_{b_k}(q_kn) = sum_j 2^(7-j) sum_{k : b_k > j} x_k bit_j(q_kn)
//   y_n = sum_g [ s_gn * ( P_gn + Phi_g ) + z_gn * X_g ],  Phi_g = sum_{k in g} x_k phi_{b_k},
//   X_g = sum_{k in g, b_k > 0} x_k.
int orc_vmm_planewise(const uint16_t* x, int T, int K, int N, int G, const uint32_t* planes, const uint16_t* scales,
                      const uint16_t* zeros, const uint8_t* bits, double* y) {
    const size_t words = (size_t)N / 32;
    const size_t plane_stride = (size_t)K * words;
    std::vector<double> P(N);
    for (int t = 0; t < T; ++t) {
        for (int n = 0; n < N; ++n) y[(size_t)t * N + n] = 0.0;
        for (int g = 0; g < K / G; ++g) {
            std::fill(P.begin(), P.end(), 0.0);
            double Phi = 0.0, X = 0.0;
            for (int i = 0; i < G; ++i) {
                int k = g * G + i;
                int b = bits[(size_t)t * K + k];
                if (b == 0) continue;
                double xv = (double)half_to_float(x[(size_t)t * K + k]);
                Phi += xv * (double)phi_of(b);
                X += xv;
            }
            for (int j = 0; j < 8; ++j) {
                double wgt = (double)(1 << (7 - j));
                for (int i = 0; i < G; ++i) {
                    int k = g * G + i;
                    if (bits[(size_t)t * K + k] <= j) continue;
                    double xv = (double)half_to_float(x[(size_t)t * K + k]) * wgt;
                    const uint32_t* row = planes + (size_t)j * plane_stride + (size_t)k * words;
                    for (int n = 0; n < N; ++n)
                        if ((row[n >> 5] >> (n & 31)) & 1u) P[n] += xv;
                }
            }
            for (int n = 0; n < N; ++n) {
                double s = (double)half_to_float(scales[(size_t)g * N + n]);
                double z = (double)half_to_float(zeros[(size_t)g * N + n]);
                y[(size_t)t * N + n] += s * (P[n] + Phi) + z * X;
            }
        }
    }
    return 0;
}

// dequantised weights at a uniform width b (test helper): w_hat[k][n] = s * code'(q, b) + z, fp64; b = 0 -> 0.
int orc_dequant(const uint32_t* planes, const uint16_t* scales, const uint16_t* zeros, int K, int N, int G, int b,
                double* w_hat) {
    for (int k = 0; k < K; ++k)
        for (int n = 0; n < N; ++n) {
            if (b == 0) {
                w_hat[(size_t)k * N + n] = 0.0;
                continue;
            }
            int q = code_from_planes(planes, K, N, k, n, b);
            double s = (double)half_to_float(scales[(size_t)(k / G) * N + n]);
            double z = (double)half_to_float(zeros[(size_t)(k / G) * N + n]);
            w_hat[(size_t)k * N + n] = s * (double)code_prime(q, b) + z;
        }
    return 0;
}

// ---- 8f2 entry points (2-bit segments, bmax in {4, 6, 8})
int orc_code2_prime(int q, int b, int bmax) { return code2_prime(q, b, bmax); }

// Quantiser of orc_pack with 2^bmax - 1 steps (reading #8), codes split into bmax / 2 segment arrays.
int orc_pack2(const uint16_t* W, int K, int N, int G, int bmax, uint32_t* segs, uint16_t* scales, uint16_t* zeros) {
    if (K % G || N % 16 || (bmax != 4 && bmax != 6 && bmax != 8)) return -2;
    const size_t words = (size_t)N / 16;
    const size_t seg_stride = (size_t)K * words;
    const float qmax = (float)((1 << bmax) - 1);
    std::memset(segs, 0, sizeof(uint32_t) * (bmax / 2) * seg_stride);
    for (int g = 0; g < K / G; ++g) {
        for (int n = 0; n < N; ++n) {
            float lo = half_to_float(W[(size_t)(g * G) * N + n]);
            float hi = lo;
            uint16_t lo_bits = W[(size_t)(g * G) * N + n];
            for (int i = 1; i < G; ++i) {
                uint16_t hb = W[(size_t)(g * G + i) * N + n];
                float v = half_to_float(hb);
                if (v < lo) {
                    lo = v;
                    lo_bits = hb;
                }
                if (v > hi) hi = v;
            }
            if (lo == 0.0f) lo_bits = 0;
            volatile float range = hi - lo;
            volatile float s32 = range / qmax;
            uint16_t s_bits = float_to_half(s32);
            float s = half_to_float(s_bits);
            float z = half_to_float(lo_bits);
            scales[(size_t)g * N + n] = s_bits;
            zeros[(size_t)g * N + n] = lo_bits;
            for (int i = 0; i < G; ++i) {
                int k = g * G + i;
                int q = 0;
                if (s != 0.0f) {
                    volatile float d = half_to_float(W[(size_t)k * N + n]) - z;
                    volatile float t = d / s;
                    float r = std::nearbyintf(t);
                    if (r < 0.0f) r = 0.0f;
                    if (r > qmax) r = qmax;
                    q = (int)r;
                }
                for (int sg = 0; sg < bmax / 2; ++sg) {
                    uint32_t pair = (uint32_t)(q >> (bmax - 2 - 2 * sg)) & 3u;
                    segs[(size_t)sg * seg_stride + (size_t)k * words + (size_t)(n >> 4)] |= pair << (2 * (n & 15));
                }
            }
        }
    }
    return 0;
}

int orc_codes2(const uint32_t* segs, int K, int N, int bmax, uint8_t* q) {
    for (int k = 0; k < K; ++k)
        for (int n = 0; n < N; ++n) q[(size_t)k * N + n] = (uint8_t)code_from_segs(segs, K, N, k, n, bmax, bmax);
    return 0;
}

// y[t][n] = sum_{k : b_tk > 0} x_tk ( s_gn code2'(q_kn, b_tk) + z_gn )  — PAPER.md:85 with the store's own bmax
int orc_vmm2_cols(const uint16_t* x, int T, int K, int N, int G, int bmax, const uint32_t* segs, const uint16_t* scales,
                  const uint16_t* zeros, const uint8_t* bits, const int32_t* cols, int ncols, double* y) {
    for (size_t i = 0; i < (size_t)T * K; ++i)
        if (bits[i] > bmax || (bits[i] & 1)) return -2;  // widths are 0, 2, .., bmax
    for (int t = 0; t < T; ++t) {
        for (int c = 0; c < ncols; ++c) {
            int n = cols ? cols[c] : c;
            double acc = 0.0;
            for (int k = 0; k < K; ++k) {
                int b = bits[(size_t)t * K + k];
                if (b == 0) continue;
                int g = k / G;
                int q = code_from_segs(segs, K, N, k, n, b, bmax);
                double s = (double)half_to_float(scales[(size_t)g * N + n]);
                double z = (double)half_to_float(zeros[(size_t)g * N + n]);
                acc += (double)half_to_float(x[(size_t)t * K + k]) * (s * (double)code2_prime(q, b, bmax) + z);
            }
            y[(size_t)t * ncols + c] = acc;
        }
    }
    return 0;
}

int orc_dequant2(const uint32_t* segs, const uint16_t* scales, const uint16_t* zeros, int K, int N, int G, int bmax,
                 int b, double* w_hat) {
    if (b > bmax || (b & 1)) return -2;
    for (int k = 0; k < K; ++k)
        for (int n = 0; n < N; ++n) {
            if (b == 0) {
                w_hat[(size_t)k * N + n] = 0.0;
                continue;
            }
            int q = code_from_segs(segs, K, N, k, n, b, bmax);
            double s = (double)half_to_float(scales[(size_t)(k / G) * N + n]);
            double z = (double)half_to_float(zeros[(size_t)(k / G) * N + n]);
            w_hat[(size_t)k * N + n] = s * (double)code2_prime(q, b, bmax) + z;
        }
    return 0;
}

}  // extern "C"
