// qw_step_stream2d.cuh — streaming temporally blocked 2D step: K applications of U = S (C (x) I)
// (eq. 7 with the shift of PAPER.md:88 eq. 8) per HBM round trip, uniform coin, natural lattice.
// Included by one translation unit per dtype.
//
// Every WARP works alone (no barrier, no shared-memory exchange between warps).  A warp owns a STRIP of HN = 32*RN
// columns (lane l: columns l*RN .. l*RN+RN-1) and streams DOWN the rows of a segment of that strip.  In its registers
// it keeps, for every time level 1 .. K, the one row of that level that is still incomplete: a pipeline of K coin
// applications through which every row passes once.  With row r of level 0 (the input) arriving,
//     level l (l = 0 .. K-1) applies the coin (eq. 1) to its row r - l, which the level below has just completed, and
//     hands the four components on to level l + 1 (eq. 8):   phi_1 -> row r-l+1   (parked until that row completes)
//                                                             phi_0 -> row r-l, one column to the right (lane shuffle)
//                                                             phi_3 -> row r-l, one column to the left  (lane shuffle)
//                                                             phi_2 -> row r-l-1: its last missing component
//     so row r-l-1 of level l+1 is complete and level l+1 goes on with it; level K's row r-K is the output row.
// The shift along m is therefore a matter of WHEN a register is consumed (no data moves, no halo along m, no
// synchronisation); only the shift along n crosses lanes: 2 complex shuffles per level and row.  The unknown outside
// of a strip travels one column per level, so the K outermost columns on each side are a halo (valid = HN - 2K).
// A segment of rows [a, b) is fed rows a-K .. b+K-1 (the pipeline fills and drains over 2K rows).
//
// The coin runs in two stages (front / back butterfly, coin_front / coin_back below) so that a level's parked registers
// are read for the last time BEFORE the level below writes its results into them: no register copies, fixed register
// roles across the back edge of the row loop (which always runs two cascades per trip).
//
// Memory: each lane copies its own 16-byte pieces of the next input rows into a per-warp ring in shared memory with
// cp.async (several rows ahead) and reads them back itself, so there is no cross-lane dependency; the row after the
// current one is already in registers; output rows go from registers to global memory as 16-byte stores.
// Work units = (walk, segment of rows, strip), strips fastest, round-robin over the warps of the persistent grid; units
// outside the light-cone diamond are skipped.
//
// Halos / walls: open lattice = broken outward links (PAPER.md:94-101 with RBL = 0): the outgoing component stays on
// its site with the opposite coin (3 - c); what lies outside the lattice is a don't-care.  Torus: the units at the seams
// wrap their input rows and columns themselves when the rows have even length (Stream2dArgs::wrap), else the halos come
// from the ghost ring of the state buffers (refreshed before the launch).  Only EDGE units (walls, seams, a lane segment
// cut by the end of the rows) run the instance with that code and with element-wise stores.
//
// Random broken links (RBL instances; eqs. 9-10, R27): level l = step t + l; one Philox call per
// lane, level and row for the four links its two sites own — see level_step.
// The deep pipeline (k = 10) parks the phi_1 rows of its first levels in shared memory (S2dShape::NS).
#pragma once

#include <type_traits>

#include "qw_coin.cuh"
#include "qw_philox.cuh"

#ifndef QW_S2D_WAVE
#define QW_S2D_WAVE 0
#endif

namespace qw {

// Launch shape per dtype and block depth K: RN = columns per lane (strip of 32*RN columns; a lane's row segment is a
// whole number of 16-byte vectors), WPC = warps per CTA (one CTA per SM; 12 warps leave 168 registers per thread, 8 leave
// 255 — the pipeline holds 4*RN complex amplitudes per level), RING / PF = rows of the per-warp input ring in shared
// memory / prefetch distance (WPC * RING * 4 * 32*RN * sizeof(complex) <= 192 KiB).
template <typename R, int K, bool RBL = false> struct S2dShape;
// NS = number of levels (the first NS) whose two parked phi_1 rows live in shared memory instead of registers (one 16-byte
// load and store per level and row): what lets the deep pipelines fit the register file.
#ifndef QW_S2D_NS10
#define QW_S2D_NS10 5
#endif
template <int K, bool RBL> struct S2dShape<float, K, RBL> {      // (link draws cost ~25 registers: 8 warps from k = 4 on)
    static constexpr int RN = 2, WPC = (K <= (RBL ? 2 : 4)) ? 12 : 8, RING = 8, PF = 6;
    static constexpr int NS = K <= 8 ? 0 : QW_S2D_NS10;
    // two rows per trip as a wavefront (cascade2): the default depth only (+1.5 % on K3; it doubles the compile time of an instance)
    static constexpr bool WAVE = QW_S2D_WAVE != 0 || (K == 8 && !RBL);
};
// (complex128 with 64-column strips at k >= 6 — all phi_1 rows in shared memory — was measured and dropped: 1.25e11 against
// 2.3e11 site-updates/s on the K2 lattice; two 32-byte shared-memory round trips per level and row bind the load/store pipe.)
template <int K, bool RBL> struct S2dShape<double, K, RBL> {
    static constexpr int RN = (K <= 4) ? 2 : 1, WPC = (K <= (RBL ? 0 : 2)) ? 12 : 8, RING = (K <= 4) ? 4 : 8, PF = RING - 1;
    static constexpr int NS = 0;
    static constexpr bool WAVE = QW_S2D_WAVE != 0;
};

template <typename R>
struct Stream2dArgs {
    const typename Cx<R>::T *in;  // site (0,0) of walk 0, plane 0 of the input buffer
    typename Cx<R>::T *out;       // ... of the output buffer
    long long em, en, pitch, walk_stride, plane_stride;
    long long max_col;            // largest column index a lane may address (row allocation end), a multiple of RN
    int wrap;                     // torus without the ghost ring: the units at the seams wrap their input rows / columns
                                  // themselves (rows of even length: lane segments stay whole and aligned)
    int batch;
    int strip0, strips;           // launched range of the global strip grid: strip j owns columns [j*V, (j+1)*V)
    long long row_lo, row_hi;     // launched rows (inclusive), cut into `segs` segments of `seg_len` rows
    long long seg_len;
    int segs;
    long long units;              // batch * segs * strips
    R coin[32];
    R coin_last[32];              // deferred scale of the named coins: coin * scale^(K-1) (qw_coin.cuh: apply_coin_bare)
    R ratio;                      // Grover-like: (d - g) / g
    long long dia_m, dia_n, dia_r;   // light-cone diamond (dia_r < 0: none), as in qw_step_tiled2d.cuh
    // random broken links (RBL instances): link number = owner * 2 + axis is broken at step t iff
    // philox4x32_10(counter = (number / 4 lo, hi, t, walk), key)[number mod 4] < rbl_thr
    unsigned rbl_key0, rbl_key1, t;
    unsigned long long rbl_thr;
};

namespace s2d {

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void cp_async16_s(uint32_t dst, const void *src) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

template <typename R> __device__ __forceinline__ cplx<R> shfl_up1(cplx<R> v) {
    v.re = __shfl_up_sync(0xffffffffu, v.re, 1);
    v.im = __shfl_up_sync(0xffffffffu, v.im, 1);
    return v;
}
template <typename R> __device__ __forceinline__ cplx<R> shfl_down1(cplx<R> v) {
    v.re = __shfl_down_sync(0xffffffffu, v.re, 1);
    v.im = __shfl_down_sync(0xffffffffu, v.im, 1);
    return v;
}

// A lane's row segment of RN consecutive sites <-> 16-byte vectors
template <int RN> __device__ __forceinline__ void load_seg(const float2 *src, cplx<float> (&dst)[RN]) {
    static_assert(RN % 2 == 0, "complex64 segments are moved as float4");
#pragma unroll
    for (int q = 0; q < RN / 2; ++q) {
        const float4 v = *reinterpret_cast<const float4 *>(src + 2 * q);
        dst[2 * q] = cplx<float>{v.x, v.y};
        dst[2 * q + 1] = cplx<float>{v.z, v.w};
    }
}
template <int RN> __device__ __forceinline__ void load_seg(const double2 *src, cplx<double> (&dst)[RN]) {
#pragma unroll
    for (int j = 0; j < RN; ++j) { const double2 v = src[j]; dst[j] = cplx<double>{v.x, v.y}; }
}
template <int RN> __device__ __forceinline__ void store_seg(float2 *dst, const cplx<float> (&src)[RN]) {
#pragma unroll
    for (int q = 0; q < RN / 2; ++q)
        *reinterpret_cast<float4 *>(dst + 2 * q) = make_float4(src[2 * q].re, src[2 * q].im, src[2 * q + 1].re, src[2 * q + 1].im);
}
template <int RN> __device__ __forceinline__ void store_seg(double2 *dst, const cplx<double> (&src)[RN]) {
#pragma unroll
    for (int j = 0; j < RN; ++j) dst[j] = make_double2(src[j].re, src[j].im);
}

// What level l+1 holds of its incomplete rows between two cascades (q = the row level l coins next):
//   c0, c3   of row q-1 (already shifted along n)     c1[p]   of row q-1     c1[p^1]   of row q     (p = parity of the cascade)
template <typename R, int RN> struct Level { cplx<R> c0[RN], c3[RN], c1[2][RN]; };
template <typename R, int RN> struct Row { cplx<R> c[4][RN]; };      // the four components of a lane's row segment

// The coin in two stages, so that a level's parked registers can be REUSED IN PLACE: the front stage reads the four
// components of a site and leaves four intermediates, the back stage turns them into phi_0 .. phi_3.  For the radix-2
// coins (H (x) H, DFT) these are the two butterfly levels of qw_coin.cuh — the same operations in the same order, so the
// results are bit for bit those of apply_coin_bare / apply_coin; the other coins are evaluated completely by the front stage.
template <typename R, int KIND, bool LAST>
__device__ __forceinline__ void coin_front(const R *C, const R *Clast, R ratio, const cplx<R> (&v)[4], cplx<R> (&t)[4]) {
    if constexpr (KIND == COIN_HXH4 && !LAST) {
        t[0] = cx_add(v[0], v[1]); t[1] = cx_sub(v[0], v[1]); t[2] = cx_add(v[2], v[3]); t[3] = cx_sub(v[2], v[3]);
    } else if constexpr (KIND == COIN_HXH4 && LAST) {
        const R h = Clast[0];
        const cplx<R> s1 = cx_scale(h, v[1]), s3 = cx_scale(h, v[3]);
        t[0] = cx_fma_r(h, v[0], s1); t[1] = cx_fms_r(h, v[0], s1); t[2] = cx_fma_r(h, v[2], s3); t[3] = cx_fms_r(h, v[2], s3);
    } else if constexpr (KIND == COIN_DFT4 && !LAST) {
        t[0] = cx_add(v[0], v[2]); t[1] = cx_sub(v[0], v[2]); t[2] = cx_add(v[1], v[3]); t[3] = cx_muli(cx_sub(v[1], v[3]));
    } else if constexpr (KIND == COIN_DFT4 && LAST) {
        const R h = Clast[0];
        const cplx<R> s2 = cx_scale(h, v[2]), s3 = cx_scale(h, v[3]);
        t[0] = cx_fma_r(h, v[0], s2); t[1] = cx_fms_r(h, v[0], s2); t[2] = cx_fma_r(h, v[1], s3); t[3] = cx_muli(cx_fms_r(h, v[1], s3));
    } else {
#pragma unroll
        for (int a = 0; a < 4; ++a) t[a] = v[a];
        if constexpr (KIND == COIN_GENERAL) apply_coin<R, 4, KIND>(C, t);
        else if constexpr (LAST) apply_coin<R, 4, KIND>(Clast, t);
        else apply_coin_bare<R, KIND>(ratio, t);
    }
}
template <typename R, int KIND, int A>
__device__ __forceinline__ cplx<R> coin_back(const cplx<R> (&t)[4]) {
    if constexpr (KIND == COIN_HXH4 || KIND == COIN_DFT4)
        return A == 0 ? cx_add(t[0], t[2]) : A == 1 ? cx_add(t[1], t[3]) : A == 2 ? cx_sub(t[0], t[2]) : cx_sub(t[1], t[3]);
    else
        return t[A];
}

// One cascade: input row r (complete, in x) passes level 0, the row it completes passes level 1, ...; emit(out) is called
// with row r-K of level K.  PAR = parity of the cascade count (which of the two phi_1 slots is due).
// Order inside a level boundary (what keeps the register allocation free of moves): phi_2 of level l first; with it the
// completed row of level l+1 goes through ITS front stage, which is the last reader of the parked registers; only then
// the back stage of level l produces phi_0, phi_1, phi_3 — straight into those registers.
// WALL: r = the input row as a row of the lattice (rows 0 / em-1 are walls), jl / jr = this lane's local column of
// lattice column 0 / en-1 (or -1).
// What a warp carries through the cascades of one unit besides the pipeline itself.
template <typename R>
struct Ctx {
    const R *C, *Clast;           // coin; coin * scale^(K-1) for the last level (deferred scale)
    R ratio;
    long long em, en;
    int jl, jr;                   // this lane's local column of lattice column 0 / en-1 (walls), or -1
    // random broken links (eqs. 9-10; R27), RBL instances only
    long long colw;               // this lane's first column as a column of the lattice (wrapped on a torus)
    unsigned k0, k1, t0, walk;    // generator key, step index of level 0, walk index
    unsigned long long thr;       // a link is broken iff its 32-bit draw is below thr
    unsigned mbits;               // per level and column: is the link to the row BELOW the last coined row broken (bit L*RN + j)
};

// ---- one level boundary of a cascade: t = front-stage values of the row (lattice row q) that level L is coining
// c1s != nullptr: the two parked phi_1 rows of this level live in shared memory, c1s[parity][lane][RN] (this lane's entry).
// RBL: every link is redrawn at every step (level L = step t0 + L).  One generator call yields the four links the lane's
// two sites own (reading R27: number = owner * 2 + axis, four consecutive numbers per call); a broken link along n keeps
// phi_0 / phi_3 on their sites with the opposite coin — for the link to the next lane the owner's bit travels with one
// more shuffle —, a broken link along m is the swap (phi_2 of this row <-> parked phi_1 of the row above) one cascade
// later, when the row below is coined: the bits wait in cx.mbits.
template <typename R, int KIND, int K, int RN, bool WALL, bool RBL, int PAR, int L, bool C1S, typename Emit>
__device__ __forceinline__ void level_step(cplx<R> (&t)[RN][4], Level<R, RN> &S, typename Cx<R>::T *c1s, Ctx<R> &cx, long long q,
                                           Emit emit) {
    constexpr int C1P = 32 * RN;                        // elements between the two parities
    if constexpr (C1S) load_seg<RN>(c1s + PAR * C1P, S.c1[PAR]);
    bool bn[RN], bm[RN];                                // links owned by the sites of row q: along n (to column +1), along m (to row +1)
    if constexpr (RBL) {
        long long qq = q;                               // the row as a row of the lattice
        if constexpr (!WALL) { if (qq < 0) qq += cx.em; else if (qq >= cx.em) qq -= cx.em; }
        const unsigned long long owner = (unsigned long long)(qq * cx.en + cx.colw);
        unsigned w[4];
        if constexpr (RN == 2) {                        // even row length, even column: the two sites share one call
            rbl_group_words(owner >> 1, cx.t0 + L, cx.walk, cx.k0, cx.k1, w);
            bn[0] = w[0] < cx.thr; bm[0] = w[1] < cx.thr; bn[1] = w[2] < cx.thr; bm[1] = w[3] < cx.thr;
        } else {
            static_assert(RN == 1 || RN == 2, "link draws are written for one or two sites per lane");
            rbl_group_words(owner >> 1, cx.t0 + L, cx.walk, cx.k0, cx.k1, w);
            const bool odd = (owner & 1ull) != 0;
            bn[0] = (odd ? w[2] : w[0]) < cx.thr; bm[0] = (odd ? w[3] : w[1]) < cx.thr;
        }
        if constexpr (WALL) {                           // links that leave the lattice belong to the wall code
#pragma unroll
            for (int j = 0; j < RN; ++j) {
                const long long cj = cx.colw + j;
                const bool in = qq >= 0 && qq < cx.em && cj >= 0 && cj < cx.en;
                bn[j] = bn[j] && in && cj < cx.en - 1;
                bm[j] = bm[j] && in && qq < cx.em - 1;
            }
        }
    }
    // ---- phi_2 of row q completes row q-1 of level L+1
    cplx<R> c2n[RN];
#pragma unroll
    for (int j = 0; j < RN; ++j) c2n[j] = coin_back<R, KIND, 2>(t[j]);
    cplx<R> y2w[RN];
    if constexpr (WALL) {
#pragma unroll
        for (int j = 0; j < RN; ++j) y2w[j] = c2n[j];
        if (q == cx.em) {                              // bottom wall: phi_1 of row em-1 (parked for row em) -> c2 of row em-1
            if constexpr (C1S) load_seg<RN>(c1s + (PAR ^ 1) * C1P, S.c1[PAR ^ 1]);
#pragma unroll
            for (int j = 0; j < RN; ++j) c2n[j] = S.c1[PAR ^ 1][j];
        }
    }
    if constexpr (RBL) {
        // links between rows q-1 and q (drawn one cascade ago): broken = phi_1 of row q-1 and phi_2 of row q stay where they are
        const unsigned prev = cx.mbits >> (L * RN);
        if constexpr (C1S) { if (prev & ((1u << RN) - 1u)) load_seg<RN>(c1s + (PAR ^ 1) * C1P, S.c1[PAR ^ 1]); }
        bool any = false;
#pragma unroll
        for (int j = 0; j < RN; ++j) {
            const bool b = (prev >> j) & 1u;
            const cplx<R> up = c2n[j], parked = S.c1[PAR ^ 1][j];
            c2n[j] = b ? parked : up;
            S.c1[PAR ^ 1][j] = b ? up : parked;
            any = any || b;
        }
        if constexpr (C1S) { if (any) store_seg<RN>(c1s + (PAR ^ 1) * C1P, S.c1[PAR ^ 1]); }
        unsigned nb = 0;
#pragma unroll
        for (int j = 0; j < RN; ++j) nb |= (bm[j] ? 1u : 0u) << j;
        cx.mbits = (cx.mbits & ~(((1u << RN) - 1u) << (L * RN))) | (nb << (L * RN));
    }
    cplx<R> tn[RN][4];
    if constexpr (L + 1 < K) {
#pragma unroll
        for (int j = 0; j < RN; ++j) {
            const cplx<R> v[4] = {S.c0[j], S.c1[PAR][j], c2n[j], S.c3[j]};
            coin_front<R, KIND, L + 2 == K>(cx.C, cx.Clast, cx.ratio, v, tn[j]);
        }
    } else {
        cplx<R> out[4][RN];
#pragma unroll
        for (int j = 0; j < RN; ++j) { out[0][j] = S.c0[j]; out[1][j] = S.c1[PAR][j]; out[2][j] = c2n[j]; out[3][j] = S.c3[j]; }
        emit(out);
    }
    // ---- phi_0, phi_1, phi_3 of row q, shifted (eq. 8), into the registers that have just been read for the last time
    cplx<R> y0[RN], y3[RN];
#pragma unroll
    for (int j = 0; j < RN; ++j) { y0[j] = coin_back<R, KIND, 0>(t[j]); y3[j] = coin_back<R, KIND, 3>(t[j]); }
#pragma unroll
    for (int j = 0; j < RN; ++j) S.c1[PAR][j] = coin_back<R, KIND, 1>(t[j]);
    if constexpr (C1S) store_seg<RN>(c1s + PAR * C1P, S.c1[PAR]);
    S.c0[0] = shfl_up1(y0[RN - 1]);                    // phi_0 of the lane to the left enters column 0
    S.c3[RN - 1] = shfl_down1(y3[0]);                  // phi_3 of the lane to the right enters column RN-1
#pragma unroll
    for (int j = 1; j < RN; ++j) { S.c0[j] = y0[j - 1]; S.c3[j - 1] = y3[j]; }
    if constexpr (RBL) {
        // broken links along n: both ends keep their outgoing component with the opposite coin
        const bool bl = __shfl_up_sync(0xffffffffu, bn[RN - 1] ? 1 : 0, 1) != 0;   // the link owned by the lane to the left
        if (bl) S.c0[0] = y3[0];
        if (bn[RN - 1]) S.c3[RN - 1] = y0[RN - 1];
#pragma unroll
        for (int j = 1; j < RN; ++j) {
            if (bn[j - 1]) { S.c0[j] = y3[j]; S.c3[j - 1] = y0[j - 1]; }
        }
    }
    if constexpr (WALL) {
        // reflecting walls (RBL = 0): the outgoing component stays with the opposite coin
#pragma unroll
        for (int j = 0; j < RN; ++j) {
            if (cx.jl == j) S.c0[j] = y3[j];           // left wall:  phi_3 -> c0 of the same site
            if (cx.jr == j) S.c3[j] = y0[j];           // right wall: phi_0 -> c3 of the same site
        }
        if (q == 0) {                                  // top wall: phi_2 -> c1 of row 0 (instead of phi_1 of row -1)
#pragma unroll
            for (int j = 0; j < RN; ++j) S.c1[PAR ^ 1][j] = y2w[j];
            if constexpr (C1S) store_seg<RN>(c1s + (PAR ^ 1) * C1P, S.c1[PAR ^ 1]);
        }
    }
    if constexpr (L + 1 < K) {
#pragma unroll
        for (int j = 0; j < RN; ++j) {
#pragma unroll
            for (int a = 0; a < 4; ++a) t[j][a] = tn[j][a];
        }
    }
}

template <typename R, int KIND, int K, int RN>
__device__ __forceinline__ void front0(const cplx<R> (&x)[4][RN], cplx<R> (&t)[RN][4], const Ctx<R> &cx) {
#pragma unroll
    for (int j = 0; j < RN; ++j) {
        const cplx<R> v[4] = {x[0][j], x[1][j], x[2][j], x[3][j]};
        coin_front<R, KIND, K == 1>(cx.C, cx.Clast, cx.ratio, v, t[j]);
    }
}

// level L's slice of the warp's shared-memory phi_1 store (levels 0 .. NS-1): c1s[level][parity][lane][RN]
template <typename R, int RN, int NS, int L> __device__ __forceinline__ typename Cx<R>::T *c1_of(typename Cx<R>::T *c1s) {
    return L < NS ? c1s + L * 2 * 32 * RN : nullptr;
}

// One cascade: input row r (complete, in x) passes level 0, the row it completes passes level 1, ...; emit(out) is called
// with row r-K of level K.  PAR = parity of the cascade count (which of the two phi_1 slots is due).
// Order inside a level boundary (what keeps the register allocation free of moves): phi_2 of level l first; with it the
// completed row of level l+1 goes through ITS front stage, which is the last reader of the parked registers; only then
// the back stage of level l produces phi_0, phi_1, phi_3 — straight into those registers.
// WALL: r = the input row as a row of the lattice (rows 0 / em-1 are walls).
template <typename R, int KIND, int K, int RN, int NS, bool WALL, bool RBL, int PAR, int L, typename Emit>
struct Levels {
    static __device__ __forceinline__ void run(cplx<R> (&t)[RN][4], Level<R, RN> (&S)[K], typename Cx<R>::T *c1s, Ctx<R> &cx,
                                               long long r, Emit emit) {
        level_step<R, KIND, K, RN, WALL, RBL, PAR, L, (L < NS)>(t, S[L], c1_of<R, RN, NS, L>(c1s), cx, r - L, emit);
        if constexpr (L + 1 < K) Levels<R, KIND, K, RN, NS, WALL, RBL, PAR, L + 1, Emit>::run(t, S, c1s, cx, r, emit);
    }
};
template <typename R, int KIND, int K, int RN, int NS, bool WALL, bool RBL, int PAR, typename Emit>
__device__ __forceinline__ void cascade(const cplx<R> (&x)[4][RN], Level<R, RN> (&S)[K], typename Cx<R>::T *c1s, Ctx<R> &cx,
                                        long long r, Emit emit) {
    cplx<R> t[RN][4];
    front0<R, KIND, K, RN>(x, t, cx);
    Levels<R, KIND, K, RN, NS, WALL, RBL, PAR, 0, Emit>::run(t, S, c1s, cx, r, emit);
}

// Two cascades as a wavefront: row r (parity PAR) runs one level ahead of row r+1 (parity PAR^1), so that at any
// time two independent dependency chains are in flight in the warp.  Level L of row r+1 reads what level L of row r
// has parked in the step before: the same order of updates as two cascades one after the other.
template <typename R, int KIND, int K, int RN, int NS, bool WALL, bool RBL, int PAR, int L, typename EmitA, typename EmitB>
struct Wave {
    static __device__ __forceinline__ void run(cplx<R> (&ta)[RN][4], cplx<R> (&tb)[RN][4], Level<R, RN> (&S)[K], typename Cx<R>::T *c1s,
                                               Ctx<R> &cx, long long r, EmitA ea, EmitB eb) {
        level_step<R, KIND, K, RN, WALL, RBL, PAR, L, (L < NS)>(ta, S[L], c1_of<R, RN, NS, L>(c1s), cx, r - L, ea);
        level_step<R, KIND, K, RN, WALL, RBL, PAR ^ 1, L - 1, (L - 1 < NS)>(tb, S[L - 1], c1_of<R, RN, NS, L - 1>(c1s), cx, r + 1 - (L - 1), eb);
        if constexpr (L + 1 < K) Wave<R, KIND, K, RN, NS, WALL, RBL, PAR, L + 1, EmitA, EmitB>::run(ta, tb, S, c1s, cx, r, ea, eb);
    }
};
// mid() is called as soon as xa has been read for the last time (the caller refills it with the row after next).
template <typename R, int KIND, int K, int RN, int NS, bool WALL, bool RBL, int PAR, typename Mid, typename EmitA, typename EmitB>
__device__ __forceinline__ void cascade2(const cplx<R> (&xa)[4][RN], const cplx<R> (&xb)[4][RN], Level<R, RN> (&S)[K],
                                         typename Cx<R>::T *c1s, Ctx<R> &cx, long long r, Mid mid, EmitA ea, EmitB eb) {
    static_assert(K >= 2, "the wavefront needs two levels");
    cplx<R> ta[RN][4], tb[RN][4];
    front0<R, KIND, K, RN>(xa, ta, cx);
    mid();
    level_step<R, KIND, K, RN, WALL, RBL, PAR, 0, (0 < NS)>(ta, S[0], c1_of<R, RN, NS, 0>(c1s), cx, r, ea);
    front0<R, KIND, K, RN>(xb, tb, cx);
    Wave<R, KIND, K, RN, NS, WALL, RBL, PAR, 1, EmitA, EmitB>::run(ta, tb, S, c1s, cx, r, ea, eb);
    level_step<R, KIND, K, RN, WALL, RBL, PAR ^ 1, K - 1, (K - 1 < NS)>(tb, S[K - 1], c1_of<R, RN, NS, K - 1>(c1s), cx, r + 1 - (K - 1), eb);
}

}  // namespace s2d

template <typename R, int K, bool RBL> constexpr size_t stream2d_smem_bytes() {
    return (size_t)S2dShape<R, K, RBL>::WPC * (S2dShape<R, K, RBL>::RING * 4 + S2dShape<R, K, RBL>::NS * 2) * (32 * S2dShape<R, K, RBL>::RN) *
           sizeof(typename Cx<R>::T);
}

template <typename R, int KIND, bool OPEN, int K, bool RBL = false>
__global__ void __launch_bounds__(S2dShape<R, K, RBL>::WPC * 32, 1)
step_stream2d_kernel(const Stream2dArgs<R> a) {
    typedef typename Cx<R>::T V;
    constexpr int RN = S2dShape<R, K, RBL>::RN, HN = 32 * RN, VN = HN - 2 * K;
    constexpr int WPC = S2dShape<R, K, RBL>::WPC, RING = S2dShape<R, K, RBL>::RING, PF = S2dShape<R, K, RBL>::PF, NS = S2dShape<R, K, RBL>::NS;
    static_assert(VN > 0, "block depth too large for the strip");
    static_assert(sizeof(V) == 16 || K % 2 == 0, "complex64 strips need an even halo (16-byte aligned lane segments)");
    static_assert(K % RN == 0, "the halo must be a whole number of lane segments");
    static_assert((RING & (RING - 1)) == 0 && PF < RING, "ring depth");

    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    V *ring = reinterpret_cast<V *>(smem_raw) + (size_t)wid * (RING * 4 * HN) + lane * RN;   // ring[slot][plane][HN], this lane's segment
    const uint32_t ring_s = s2d::smem_u32(ring);
    // this lane's entry of the warp's phi_1 store c1s[level][parity][lane][RN] (behind the rings)
    V *c1s = reinterpret_cast<V *>(smem_raw) + (size_t)WPC * (RING * 4 * HN) + (size_t)wid * (NS * 2 * HN) + lane * RN;
    const long long nwarps = (long long)gridDim.x * WPC;
    const long long per_walk = (long long)a.segs * a.strips;
    const R *C = a.coin;

    // EDGE = the unit can see a wall (open lattice) or the right end of the rows (a lane segment may be cut by column
    // en): only that instance carries the wall code and the element-wise stores.
    auto run = [&](auto edge_tag, long long w, long long a0, long long b0, long long n0) {
        constexpr bool EDGE = decltype(edge_tag)::value;
        constexpr bool WALL = EDGE && OPEN;
        constexpr uint32_t PLB = HN * sizeof(V), SLOTB = 4 * PLB;             // bytes of a plane row / of a ring slot
        const long long col = n0 + lane * RN;
        long long lcol = col;
        long long row0 = a0 - K;                                               // input row a0-K comes first
        int fseam = -1;                                                        // fetches until the input rows wrap around (torus)
        if constexpr (EDGE && !OPEN) {
            if (a.wrap) {                                                      // no ghost ring: wrap rows and columns here
                if (lcol < 0) lcol += a.en; else if (lcol >= a.en) lcol -= a.en;
                if (row0 < 0) row0 += a.em;
                fseam = (int)(a.em - row0);
            }
        }
        if (lcol > a.max_col) lcol = a.max_col;                                // lanes beyond the row allocation re-read its end
        // running byte pointers (plane 0): the next input row to fetch, the next output row to store
        const char *gp = reinterpret_cast<const char *>(a.in + w * a.walk_stride + row0 * a.pitch + lcol);
        char *op = reinterpret_cast<char *>(a.out + w * a.walk_stride + a0 * a.pitch + col);
        const long long planeb = a.plane_stride * (long long)sizeof(V);
        const long long rowb = a.pitch * (long long)sizeof(V);
        const long long jl_ = -col, jr_ = a.en - 1 - col;
        s2d::Ctx<R> cx;
        cx.C = C; cx.Clast = a.coin_last; cx.ratio = a.ratio; cx.em = a.em; cx.en = a.en;
        cx.jl = (jl_ >= 0 && jl_ < RN) ? (int)jl_ : -1; cx.jr = (jr_ >= 0 && jr_ < RN) ? (int)jr_ : -1;
        if constexpr (RBL) {
            cx.colw = col;
            if constexpr (!OPEN) { if (cx.colw < 0) cx.colw += a.en; else if (cx.colw >= a.en) cx.colw -= a.en; }
            cx.k0 = a.rbl_key0; cx.k1 = a.rbl_key1; cx.t0 = a.t; cx.walk = (unsigned)w; cx.thr = a.rbl_thr; cx.mbits = 0;
        }
        const bool st_lane = (lane * RN >= K) && (lane * RN + RN <= HN - K) && col < a.en;
        const bool st_full = col + RN <= a.en;                                 // always true in a unit that is not EDGE
        const int nrows = (int)(b0 - a0) + 2 * K;
        uint32_t fslot = 0, lslot = 0;                                         // ring slot offsets (bytes) of the next fetch / next read
        int fleft = nrows;                                                     // input rows not yet fetched

        s2d::Level<R, RN> S[K];
#pragma unroll
        for (int l = 0; l < K; ++l) {
#pragma unroll
            for (int j = 0; j < RN; ++j)
                S[l].c0[j] = S[l].c3[j] = S[l].c1[0][j] = S[l].c1[1][j] = cplx<R>{0, 0};
        }
#pragma unroll
        for (int l = 0; l < 2 * NS; ++l) s2d::store_seg<RN>(c1s + l * HN, S[0].c0);
        auto fetch = [&]() {                       // the next input row -> the next ring slot
            if (fleft > 0) {
                const char *g = gp;
#pragma unroll
                for (int c = 0; c < 4; ++c) {
#pragma unroll
                    for (int q = 0; q < (int)(RN * sizeof(V) / 16); ++q)
                        s2d::cp_async16_s(ring_s + fslot + c * PLB + 16 * q, g + 16 * q);
                    g += planeb;
                }
                gp += rowb;
                if constexpr (EDGE && !OPEN) { if (--fseam == 0) { gp -= a.em * rowb; fseam = (int)a.em; } }   // (a unit may cross both seams)
            }
            --fleft;
            fslot = (fslot + SLOTB) & (RING * SLOTB - 1);
            s2d::cp_async_commit();
        };
        auto take = [&](s2d::Row<R, RN> &x) {      // the next ring slot -> registers (the lane reads what it copied itself)
            const V *sl = reinterpret_cast<const V *>(reinterpret_cast<const char *>(ring) + lslot);
            lslot = (lslot + SLOTB) & (RING * SLOTB - 1);
#pragma unroll
            for (int c = 0; c < 4; ++c) s2d::load_seg<RN>(sl + c * HN, x.c[c]);
        };
        // the output row of input row i: a0 + (i - 2K)
        auto put = [&](int i, const cplx<R> (&o)[4][RN]) {
            const bool row_ok = i >= 2 * K && i < nrows;
            if (row_ok && st_lane && (!EDGE || st_full)) {
                char *o_ = op;
#pragma unroll
                for (int c = 0; c < 4; ++c) { s2d::store_seg<RN>(reinterpret_cast<V *>(o_), o[c]); o_ += planeb; }
            }
            if constexpr (EDGE) {
                if (row_ok && st_lane && !st_full) {
                    char *o_ = op;
#pragma unroll
                    for (int c = 0; c < 4; ++c) {
#pragma unroll
                        for (int j = 0; j < RN; ++j)
                            if (col + j < a.en) cx_store<R>(reinterpret_cast<V *>(o_) + j, o[c][j]);
                        o_ += planeb;
                    }
                }
            }
            if (i >= 2 * K) op += rowb;
        };
#pragma unroll 1
        for (int i = 0; i < PF; ++i) fetch();
        s2d::cp_async_wait<PF - 1>();
        s2d::Row<R, RN> xa, xb;
        take(xa);
        if constexpr (S2dShape<R, K, RBL>::WAVE) {
        // two input rows per trip, their cascades interleaved as a wavefront (s2d::cascade2)
#pragma unroll 1
        for (int i = 0; i < nrows; i += 2) {       // a surplus odd row is not stored
            fetch();
            fetch();
            s2d::cp_async_wait<PF - 1>();
            take(xb);
            s2d::cascade2<R, KIND, K, RN, NS, WALL, RBL, 0>(xa.c, xb.c, S, c1s, cx, a0 - K + i,
                                                   [&]() { take(xa); },
                                                   [&](const cplx<R> (&o)[4][RN]) { put(i, o); },
                                                   [&](const cplx<R> (&o)[4][RN]) { put(i + 1, o); });
        }
        } else {
        // one cascade on x (input row i of the unit) while the row after it is taken from the ring into xn
        auto one = [&](auto par_tag, int i, const s2d::Row<R, RN> &x, s2d::Row<R, RN> &xn) {
            constexpr int PAR = decltype(par_tag)::value;
            fetch();
            s2d::cp_async_wait<PF - 1>();
            take(xn);
            s2d::cascade<R, KIND, K, RN, NS, WALL, RBL, PAR>(x.c, S, c1s, cx, a0 - K + i,
                                                    [&](const cplx<R> (&o)[4][RN]) { put(i, o); });
        };
#pragma unroll 1
        for (int i = 0; i < nrows; i += 2) {       // always two cascades per trip (fixed register roles); a surplus odd row is not stored
            one(std::integral_constant<int, 0>{}, i, xa, xb);
            one(std::integral_constant<int, 1>{}, i + 1, xb, xa);
        }
        }
        s2d::cp_async_wait<0>();
    };

    // Unit g of this warp: g = warp, warp + nwarps, ...  Without a light-cone diamond g indexes ALL units (walk, segment, strip;
    // strips fastest).  With a diamond g indexes the ACTIVE units only — in every (walk, segment) the strips that meet the
    // diamond are one interval [lo, lo + cnt), found in closed form — so that the active units, not the units of the bounding
    // box, are dealt round-robin (else a warp whose share lies outside the diamond idles: 1.5x on the K2 cone); the warp scans
    // the (walk, segment) rows once, carrying the number of active units before the current row (qbase).
    long long g = (long long)blockIdx.x * WPC + wid;
    long long qw_ = 0, qbase = 0;                  // diamond scan: walk of the current row, active units before it
    int qseg = -1, qcnt = 0, qlo = 0;              // ... its segment (-1: before the first), its active strips [qlo, qlo + qcnt)
    for (;; g += nwarps) {
        long long w, a0, b0;
        int strip;
        if (a.dia_r >= 0) {
            bool found = true;
            while (g >= qbase + qcnt) {            // advance to the row that holds active unit g
                qbase += qcnt;
                if (++qseg == a.segs) { qseg = 0; ++qw_; }
                if (qw_ >= a.batch) { found = false; break; }
                const long long ra = a.row_lo + (long long)qseg * a.seg_len;
                long long rb = ra + a.seg_len;
                if (rb > a.row_hi + 1) rb = a.row_hi + 1;
                qcnt = 0;
                if (ra < rb) {
                    const long long dm = a.dia_m < ra ? ra - a.dia_m : (a.dia_m > rb - 1 ? a.dia_m - (rb - 1) : 0);
                    const long long rem = a.dia_r - dm;          // strip j is active iff its distance along n is <= rem
                    if (rem >= 0) {
                        long long lo = (a.dia_n - rem) / VN, hi = (a.dia_n + rem) / VN;   // (strip0 >= 0 absorbs the rounding of negatives)
                        if (lo < a.strip0) lo = a.strip0;
                        if (hi > a.strip0 + a.strips - 1) hi = a.strip0 + a.strips - 1;
                        if (hi >= lo) { qlo = (int)lo; qcnt = (int)(hi - lo + 1); }
                    }
                }
            }
            if (!found) break;
            w = qw_;
            strip = qlo + (int)(g - qbase);
            a0 = a.row_lo + (long long)qseg * a.seg_len;
            b0 = a0 + a.seg_len;
            if (b0 > a.row_hi + 1) b0 = a.row_hi + 1;
        } else {
            if (g >= a.units) break;
            w = g / per_walk;
            const long long rr = g - w * per_walk;
            const int seg = (int)(rr / a.strips);
            strip = a.strip0 + (int)(rr - (long long)seg * a.strips);
            a0 = a.row_lo + seg * a.seg_len;
            b0 = a0 + a.seg_len;
            if (b0 > a.row_hi + 1) b0 = a.row_hi + 1;
            if (a0 >= b0) continue;
        }
        const long long n_lo = (long long)strip * VN, n0 = n_lo - K;
        bool edge = n0 + HN >= a.en;               // the strip holds the right end of the rows
        if constexpr (!OPEN) edge = edge || (a.wrap && (a0 - K < 0 || b0 + K + 1 > a.em || n0 < 0));   // ... or a seam of the torus
        if constexpr (OPEN) edge = edge || (a0 - K <= 0) || (b0 + K >= a.em) || (n0 <= 0);
        if (edge) run(std::true_type{}, w, a0, b0, n0);
        else run(std::false_type{}, w, a0, b0, n0);
    }
}

}  // namespace qw
