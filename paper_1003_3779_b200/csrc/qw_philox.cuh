// qw_philox.cuh — the counter-based generator of the random-broken-links model (eqs. 9-10;
// DESIGN.md reading R27), device side.  Shared by the step kernels of libqw only; the oracle has its own copy.
#pragma once

namespace qw {

// Philox4x32-10 (Salmon, Moraes, Dror, Shaw, "Parallel random numbers: as easy as 1, 2, 3", SC'11), written from the
// published round function: all four output words.
__device__ __forceinline__ void philox4x32_10(unsigned c0, unsigned c1, unsigned c2, unsigned c3, unsigned k0, unsigned k1,
                                              unsigned (&w)[4]) {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const unsigned long long p0 = (unsigned long long)0xD2511F53u * c0, p1 = (unsigned long long)0xCD9E8D57u * c2;
        const unsigned hi0 = (unsigned)(p0 >> 32), lo0 = (unsigned)p0, hi1 = (unsigned)(p1 >> 32), lo1 = (unsigned)p1;
        c0 = hi1 ^ c1 ^ k0; c1 = lo1; c2 = hi0 ^ c3 ^ k1; c3 = lo0;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    w[0] = c0; w[1] = c1; w[2] = c2; w[3] = c3;
}

// The link function of reading R27: links are numbered owner * dim + axis; the call with counter
// (number / 4, t, walk) yields the states of the four links 4g .. 4g+3, one per output word.
__device__ __forceinline__ void rbl_group_words(unsigned long long group, unsigned t, unsigned walk, unsigned k0, unsigned k1,
                                                unsigned (&w)[4]) {
    philox4x32_10((unsigned)group, (unsigned)(group >> 32), t, walk, k0, k1, w);
}
__device__ __forceinline__ unsigned rbl_link_word(unsigned long long number, unsigned t, unsigned walk, unsigned k0, unsigned k1) {
    unsigned w[4];
    rbl_group_words(number >> 2, t, walk, k0, k1, w);
    const unsigned sel = (unsigned)number & 3u;
    return sel == 0 ? w[0] : (sel == 1 ? w[1] : (sel == 2 ? w[2] : w[3]));
}

}  // namespace qw
