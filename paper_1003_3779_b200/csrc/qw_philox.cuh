// qw_philox.cuh — the counter-based generator of the random-broken-links model (eqs. 9-10;
// DESIGN.md reading R27), device side.  Shared by the step kernels of libqw only; the oracle has its own copy.
#pragma once

namespace qw {

// Philox4x32-10 (Salmon, Moraes, Dror, Shaw, "Parallel random numbers: as easy as 1, 2, 3", SC'11), written from the
// published round function.  Returns output word `axis` (0 or 1).
__device__ __forceinline__ unsigned philox4x32_10_word(unsigned c0, unsigned c1, unsigned c2, unsigned c3,
                                                       unsigned k0, unsigned k1, int axis) {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const unsigned hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
        const unsigned hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
        c0 = hi1 ^ c1 ^ k0; c1 = lo1; c2 = hi0 ^ c3 ^ k1; c3 = lo0;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    return axis == 0 ? c0 : c1;
}

// Both words of one call: the states of the two links a site OWNS (axis 0 and axis 1).
__device__ __forceinline__ void philox4x32_10_words01(unsigned c0, unsigned c1, unsigned c2, unsigned c3,
                                                      unsigned k0, unsigned k1, unsigned &w0, unsigned &w1) {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const unsigned hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
        const unsigned hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
        c0 = hi1 ^ c1 ^ k0; c1 = lo1; c2 = hi0 ^ c3 ^ k1; c3 = lo0;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    w0 = c0; w1 = c1;
}

}  // namespace qw
