// qw_step_tiled2d.cuh — register-tiled temporally blocked 2D step: K applications of
// U = S (C (x) I) (eq. 7 with the shift of PAPER.md:88 eq. 8) per HBM round trip,
// uniform coin, natural lattice.  Included by one translation unit per dtype.
//
// A persistent CTA of W warps walks over tiles of HM x HN = (W*RM) x (32*RN) sites (valid interior
// (HM-2K) x (HN-2K) plus a K-site halo: after K steps the unknown outside has travelled exactly K
// sites inwards, eq. 18).  Warp w owns the strip of RM rows w*RM .. w*RM+RM-1, lane l
// the RM x RN patch of columns l*RN .. l*RN+RN-1 of that strip, for all four coin planes, IN REGISTERS.
//
// One step:
//   coin   in place on the four registers of every site                         (eq. 1)
//   shift  (eq. 8) is a RENAMING of registers inside a patch: at step s the amplitude of logical
//          site (i, j) lives in  c0[i][(j-s) mod RN]  (moves n+1)   c1[(i-s) mod RM][j]  (moves m+1)
//                                c3[i][(j+s) mod RN]  (moves n-1)   c2[(i+s) mod RM][j]  (moves m-1)
//          so only what crosses a patch edge moves: per step RM elements of c0 / c3 go to the
//          neighbouring lane through warp shuffles and RN elements of c1 / c2 go to the neighbouring
//          warp through a double-buffered shared-memory slot guarded by one mbarrier per warp: a
//          warp waits for its two neighbours only, never for the whole CTA.
//          The K steps are fully unrolled, so every register index is a compile-time constant.
//   walls  (open lattice = broken outward links, PAPER.md:94-101 with RBL = 0): at a wall site the
//          outgoing component overrides what would have come in from outside, with the opposite
//          coin (3-c).  Sites outside the lattice compute don't-care values that never enter.
//
// Memory: the next tile of the CTA is prefetched by TMA (cp.async.bulk.tensor + mbarrier) into a
// shared-memory stage while the current one is advanced in registers; the stage is drained into
// registers at the start of the tile (it is free again at once), results go from registers
// straight to global memory.  Halos come from the ghost ring of the state buffers (periodic:
// refreshed before each launch; open: zeros); beyond the allocation TMA zero-fills.
#pragma once

#include <cuda.h>

#include "qw_coin.cuh"

namespace qw {

template <typename R> struct T2dCfg;
#ifndef QW_T2D_F32_RM
#define QW_T2D_F32_RM 4
#define QW_T2D_F32_W 16
#define QW_T2D_F32_NSYNC false
#endif
template <> struct T2dCfg<float>  { static constexpr int RM = QW_T2D_F32_RM, RN = 2, W = QW_T2D_F32_W; static constexpr bool NSYNC = QW_T2D_F32_NSYNC; };  // 64 x 64 sites, 128 KiB stage
#ifndef QW_T2D_F64_RM
#define QW_T2D_F64_RM 4
#define QW_T2D_F64_W 8
#define QW_T2D_F64_NSYNC true
#endif
template <> struct T2dCfg<double> { static constexpr int RM = QW_T2D_F64_RM, RN = 2, W = QW_T2D_F64_W;  static constexpr bool NSYNC = QW_T2D_F64_NSYNC; };   // 32 x 64 sites, 128 KiB stage

template <typename R>
struct Tiled2dArgs {
    typename Cx<R>::T *out;       // site (0,0) of walk 0, plane 0 of the output buffer
    long long em, en, pitch, walk_stride, plane_stride;
    long long total_tiles;        // tiles_m * tiles_n * batch
    int batch, ghost;
    int tile_m0, tile_n0;         // first tile (of the global tile grid) of the launched range
    int tiles_m, tiles_n;         // extent of the launched range
    R coin[32];
    // deferred scale of the named coins (qw_coin.cuh: apply_coin_bare): steps 0 .. K-2 run the bare coin, step K-1
    // the scaled evaluation with coin_last = coin * scale^(K-1) (an exact power-of-two multiple)
    R coin_last[32];
    R ratio;                      // Grover-like: (d - g) / g
    // light-cone DIAMOND (natural lattice: every step moves one site along one axis, so after t steps a delta start
    // is confined to |m - m0| + |n - n0| <= t): tiles whose output sites all lie outside it are
    // skipped (they are exact zeros in both buffers).  dia_r < 0: no diamond, every tile of the range is computed.
    long long dia_m, dia_n, dia_r;
};

__host__ __device__ constexpr int t2d_mod(int a, int m) { return ((a % m) + m) % m; }

namespace t2d {

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t *bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity) {
    uint32_t done;
    do {
        asm volatile(
            "{\n\t.reg .pred p;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t}"
            : "=r"(done) : "r"(smem_u32(bar)), "r"(parity) : "memory");
    } while (!done);
}
__device__ __forceinline__ void tma_load_3d(void *dst, const CUtensorMap *map, int c0, int c1, int c2, uint64_t *bar) {
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
        ::"r"(smem_u32(dst)), "l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(smem_u32(bar)) : "memory");
}

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

template <typename R> __device__ __forceinline__ typename Cx<R>::T make_v(cplx<R> z) {
    typename Cx<R>::T v; v.x = z.re; v.y = z.im; return v;
}

// A lane's row segment of RN consecutive sites: 16-byte vector accesses (shared or global memory).
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

// The register patch of one lane: four coin planes of RM x RN sites.
template <typename R, int RM, int RN>
struct Patch {
    cplx<R> c0[RM][RN], c1[RM][RN], c2[RM][RN], c3[RM][RN];
};

// Where the lattice walls cut this lane's patch (local row / column index, or -1).
struct Walls {
    int il, ir;   // local row of lattice row 0 / em-1 inside this warp's strip
    int jl, jr;   // local column of lattice column 0 / en-1 inside this lane's patch
};

// One walk step, S = number of steps already applied to this tile (compile time).
// xb = exchange slots of this step's parity: V xb[W][2][RN][32]; xbar = their W "slot of warp w is full"
// mbarriers; bit (S & 1) of xph = the phase parity to wait for.  A warp only waits for its two neighbours:
// they can never be more than one step apart, so the double-buffered slots and barriers are race-free.
template <typename R, int RM, int RN, int W, int KIND, bool OPEN, int S, bool LAST>
__device__ __forceinline__ void step(Patch<R, RM, RN> &p, const R *C, const R *Clast, R ratio, typename Cx<R>::T *xb,
                                     uint64_t *xbar, uint32_t &xph, int lane, int wid, bool wall_tile, const Walls &wl) {
    typedef typename Cx<R>::T V;
    // ---- coin (eq. 1) on every site of the patch, in place
#pragma unroll
    for (int i = 0; i < RM; ++i) {
#pragma unroll
        for (int j = 0; j < RN; ++j) {
            cplx<R> v[4] = {p.c0[i][t2d_mod(j - S, RN)], p.c1[t2d_mod(i - S, RM)][j],
                            p.c2[t2d_mod(i + S, RM)][j], p.c3[i][t2d_mod(j + S, RN)]};
            if constexpr (KIND == COIN_GENERAL) apply_coin<R, 4, KIND>(C, v);
            else if constexpr (LAST) apply_coin<R, 4, KIND>(Clast, v);
            else apply_coin_bare<R, KIND>(ratio, v);
            p.c0[i][t2d_mod(j - S, RN)] = v[0];
            p.c1[t2d_mod(i - S, RM)][j] = v[1];
            p.c2[t2d_mod(i + S, RM)][j] = v[2];
            p.c3[i][t2d_mod(j + S, RN)] = v[3];
        }
    }
    // ---- shift (eq. 8): only the patch edges move
    constexpr int Q0 = t2d_mod(RN - 1 - S, RN);   // phi_0 of logical column RN-1 -> column 0 of the lane to the right
    constexpr int P3 = t2d_mod(S, RN);            // phi_3 of logical column 0    -> column RN-1 of the lane to the left
    constexpr int Q1 = t2d_mod(RM - 1 - S, RM);   // phi_1 of logical row RM-1    -> row 0 of the warp below
    constexpr int P2 = t2d_mod(S, RM);            // phi_2 of logical row 0       -> row RM-1 of the warp above
#pragma unroll
    for (int j = 0; j < RN; ++j) {
        V z1, z2;
        z1.x = p.c1[Q1][j].re; z1.y = p.c1[Q1][j].im;
        z2.x = p.c2[P2][j].re; z2.y = p.c2[P2][j].im;
        xb[((wid * 2 + 0) * RN + j) * 32 + lane] = z1;
        xb[((wid * 2 + 1) * RN + j) * 32 + lane] = z2;
    }
    // NSYNC: neighbour-only synchronisation through mbarriers; otherwise one __syncthreads per step
    constexpr bool NSYNC = T2dCfg<R>::NSYNC;
    uint32_t par = 0;
    if constexpr (NSYNC) {
        __syncwarp();
        if (lane == 0) mbar_arrive(xbar + wid);
        par = (xph >> (S & 1)) & 1u;
        xph ^= 1u << (S & 1);
    }
    if (OPEN && wall_tile) {                       // CTA-uniform branch
        // reflecting walls (RBL = 0): the outgoing component stays with the opposite coin
        cplx<R> f1[RN], f2[RN];
#pragma unroll
        for (int j = 0; j < RN; ++j) { f1[j] = cplx<R>{0, 0}; f2[j] = cplx<R>{0, 0}; }
#pragma unroll
        for (int i = 0; i < RM; ++i) {
            if (wl.ir == i) {                      // bottom wall: phi_1 -> c2 of the same site
#pragma unroll
                for (int j = 0; j < RN; ++j) f2[j] = p.c1[t2d_mod(i - S, RM)][j];
            }
            if (wl.il == i) {                      // top wall: phi_2 -> c1 of the same site
#pragma unroll
                for (int j = 0; j < RN; ++j) f1[j] = p.c2[t2d_mod(i + S, RM)][j];
            }
        }
#pragma unroll
        for (int i = 0; i < RM; ++i) {
            const cplx<R> t0 = shfl_up1(p.c0[i][Q0]);
            const cplx<R> t3 = shfl_down1(p.c3[i][P3]);
            cplx<R> f3 = {0, 0}, f0 = {0, 0};
#pragma unroll
            for (int j = 0; j < RN; ++j) {
                if (wl.jr == j) f3 = p.c0[i][t2d_mod(j - S, RN)];    // right wall: phi_0 -> c3 of the same site
                if (wl.jl == j) f0 = p.c3[i][t2d_mod(j + S, RN)];    // left wall:  phi_3 -> c0 of the same site
            }
            p.c0[i][Q0] = t0;
            p.c3[i][P3] = t3;
#pragma unroll
            for (int j = 0; j < RN; ++j) {
                if (wl.jr == j) p.c3[i][t2d_mod(j + S + 1, RN)] = f3;
                if (wl.jl == j) p.c0[i][t2d_mod(j - S - 1, RN)] = f0;
            }
        }
        if constexpr (!NSYNC) __syncthreads();
        if (wid > 0) {
            if constexpr (NSYNC) mbar_wait(xbar + wid - 1, par);
#pragma unroll
            for (int j = 0; j < RN; ++j) p.c1[Q1][j] = cx_load<R>(xb + (((wid - 1) * 2 + 0) * RN + j) * 32 + lane);
        }
        if (wid < W - 1) {
            if constexpr (NSYNC) mbar_wait(xbar + wid + 1, par);
#pragma unroll
            for (int j = 0; j < RN; ++j) p.c2[P2][j] = cx_load<R>(xb + (((wid + 1) * 2 + 1) * RN + j) * 32 + lane);
        }
#pragma unroll
        for (int i = 0; i < RM; ++i) {
            if (wl.ir == i) {
#pragma unroll
                for (int j = 0; j < RN; ++j) p.c2[t2d_mod(i + S + 1, RM)][j] = f2[j];
            }
            if (wl.il == i) {
#pragma unroll
                for (int j = 0; j < RN; ++j) p.c1[t2d_mod(i - S - 1, RM)][j] = f1[j];
            }
        }
    } else {
#pragma unroll
        for (int i = 0; i < RM; ++i) {
            p.c0[i][Q0] = shfl_up1(p.c0[i][Q0]);
            p.c3[i][P3] = shfl_down1(p.c3[i][P3]);
        }
        if constexpr (!NSYNC) __syncthreads();
        if (wid > 0) {
            if constexpr (NSYNC) mbar_wait(xbar + wid - 1, par);
#pragma unroll
            for (int j = 0; j < RN; ++j) p.c1[Q1][j] = cx_load<R>(xb + (((wid - 1) * 2 + 0) * RN + j) * 32 + lane);
        }
        if (wid < W - 1) {
            if constexpr (NSYNC) mbar_wait(xbar + wid + 1, par);
#pragma unroll
            for (int j = 0; j < RN; ++j) p.c2[P2][j] = cx_load<R>(xb + (((wid + 1) * 2 + 1) * RN + j) * 32 + lane);
        }
    }
}

template <typename R, int RM, int RN, int W, int KIND, bool OPEN, int S, int K>
struct Steps {
    static __device__ __forceinline__ void run(Patch<R, RM, RN> &p, const R *C, const R *Clast, R ratio, typename Cx<R>::T *xch,
                                               uint64_t *xbar, uint32_t &xph, int lane, int wid, bool wall_tile, const Walls &wl) {
        step<R, RM, RN, W, KIND, OPEN, S, S + 1 == K>(p, C, Clast, ratio, xch + (S & 1) * (W * 2 * RN * 32), xbar + (S & 1) * W, xph,
                                                      lane, wid, wall_tile, wl);
        if constexpr (S + 1 < K)
            Steps<R, RM, RN, W, KIND, OPEN, S + 1, K>::run(p, C, Clast, ratio, xch, xbar, xph, lane, wid, wall_tile, wl);
    }
};

// ---------------------------------------------------------------------------------------------------------------
// DIAGONAL lattice (Fig. 1c, the lattice of the paper's Tables 2-3): component c = 2j+k moves BOTH
// coordinates, (m + (-1)^j, n + (-1)^k).  Renaming at step s: the amplitude of logical site (i, j) lives in
//     c0[(i-s) mod RM][(j-s) mod RN]   c1[(i-s) mod RM][(j+s) mod RN]
//     c2[(i+s) mod RM][(j-s) mod RN]   c3[(i+s) mod RM][(j+s) mod RN]
// Per step the edge COLUMN of every plane crosses a lane boundary (shuffles, all RM rows), then the edge ROW of every
// plane (already holding the shuffled corner element) crosses a warp boundary through the exchange slots
// xb[W][4][RN][32].  No wall code: the kernel is only launched where no amplitude can touch a wall (torus, or an
// open lattice while the light cone stays inside: the dispatcher checks it per launch).
template <typename R, int RM, int RN, int W, int KIND, int S, bool LAST>
__device__ __forceinline__ void step_diag(Patch<R, RM, RN> &p, const R *C, const R *Clast, R ratio, typename Cx<R>::T *xb,
                                          uint64_t *xbar, uint32_t &xph, int lane, int wid) {
    typedef typename Cx<R>::T V;
#pragma unroll
    for (int i = 0; i < RM; ++i) {
#pragma unroll
        for (int j = 0; j < RN; ++j) {
            const int im = t2d_mod(i - S, RM), ip = t2d_mod(i + S, RM), jm = t2d_mod(j - S, RN), jp = t2d_mod(j + S, RN);
            cplx<R> v[4] = {p.c0[im][jm], p.c1[im][jp], p.c2[ip][jm], p.c3[ip][jp]};
            if constexpr (KIND == COIN_GENERAL) apply_coin<R, 4, KIND>(C, v);
            else if constexpr (LAST) apply_coin<R, 4, KIND>(Clast, v);
            else apply_coin_bare<R, KIND>(ratio, v);
            p.c0[im][jm] = v[0]; p.c1[im][jp] = v[1]; p.c2[ip][jm] = v[2]; p.c3[ip][jp] = v[3];
        }
    }
    constexpr int QN = t2d_mod(RN - 1 - S, RN);   // column register of the planes moving n+1 (c0, c2) that leaves to the right
    constexpr int PN = t2d_mod(S, RN);            // column register of the planes moving n-1 (c1, c3) that leaves to the left
    constexpr int QM = t2d_mod(RM - 1 - S, RM);   // row register of the planes moving m+1 (c0, c1) that leaves downwards
    constexpr int PM = t2d_mod(S, RM);            // row register of the planes moving m-1 (c2, c3) that leaves upwards
    // ---- columns first (so that the corner element travels with its row afterwards)
#pragma unroll
    for (int r = 0; r < RM; ++r) {
        p.c0[r][QN] = shfl_up1(p.c0[r][QN]);
        p.c2[r][QN] = shfl_up1(p.c2[r][QN]);
        p.c1[r][PN] = shfl_down1(p.c1[r][PN]);
        p.c3[r][PN] = shfl_down1(p.c3[r][PN]);
    }
    // ---- rows through the exchange slots
#pragma unroll
    for (int j = 0; j < RN; ++j) {
        xb[((wid * 4 + 0) * RN + j) * 32 + lane] = make_v<R>(p.c0[QM][j]);
        xb[((wid * 4 + 1) * RN + j) * 32 + lane] = make_v<R>(p.c1[QM][j]);
        xb[((wid * 4 + 2) * RN + j) * 32 + lane] = make_v<R>(p.c2[PM][j]);
        xb[((wid * 4 + 3) * RN + j) * 32 + lane] = make_v<R>(p.c3[PM][j]);
    }
    constexpr bool NSYNC = T2dCfg<R>::NSYNC;
    uint32_t par = 0;
    if constexpr (NSYNC) {
        __syncwarp();
        if (lane == 0) mbar_arrive(xbar + wid);
        par = (xph >> (S & 1)) & 1u;
        xph ^= 1u << (S & 1);
    } else {
        __syncthreads();
    }
    if (wid > 0) {
        if constexpr (NSYNC) mbar_wait(xbar + wid - 1, par);
#pragma unroll
        for (int j = 0; j < RN; ++j) {
            p.c0[QM][j] = cx_load<R>(xb + (((wid - 1) * 4 + 0) * RN + j) * 32 + lane);
            p.c1[QM][j] = cx_load<R>(xb + (((wid - 1) * 4 + 1) * RN + j) * 32 + lane);
        }
    }
    if (wid < W - 1) {
        if constexpr (NSYNC) mbar_wait(xbar + wid + 1, par);
#pragma unroll
        for (int j = 0; j < RN; ++j) {
            p.c2[PM][j] = cx_load<R>(xb + (((wid + 1) * 4 + 2) * RN + j) * 32 + lane);
            p.c3[PM][j] = cx_load<R>(xb + (((wid + 1) * 4 + 3) * RN + j) * 32 + lane);
        }
    }
}

template <typename R, int RM, int RN, int W, int KIND, int S, int K>
struct StepsDiag {
    static __device__ __forceinline__ void run(Patch<R, RM, RN> &p, const R *C, const R *Clast, R ratio, typename Cx<R>::T *xch,
                                               uint64_t *xbar, uint32_t &xph, int lane, int wid) {
        step_diag<R, RM, RN, W, KIND, S, S + 1 == K>(p, C, Clast, ratio, xch + (S & 1) * (W * 4 * RN * 32), xbar + (S & 1) * W, xph,
                                                     lane, wid);
        if constexpr (S + 1 < K) StepsDiag<R, RM, RN, W, KIND, S + 1, K>::run(p, C, Clast, ratio, xch, xbar, xph, lane, wid);
    }
};

}  // namespace t2d

template <typename R, bool DIAG = false> constexpr size_t tiled2d_smem_bytes() {
    typedef T2dCfg<R> G;
    return (size_t)4 * (G::W * G::RM) * (32 * G::RN) * sizeof(typename Cx<R>::T)      // TMA stage
         + (size_t)2 * G::W * (DIAG ? 4 : 2) * G::RN * 32 * sizeof(typename Cx<R>::T) // exchange slots
         + (size_t)(2 * G::W + 2) * 8;                                                // mbarriers
}

template <typename R, int KIND, bool OPEN, int K, bool DIAG = false>
__global__ void __launch_bounds__(T2dCfg<R>::W * 32, 1)
step_tiled2d_kernel(const __grid_constant__ CUtensorMap tmap, const Tiled2dArgs<R> a) {
    typedef typename Cx<R>::T V;
    typedef T2dCfg<R> G;
    constexpr int RM = G::RM, RN = G::RN, W = G::W;
    constexpr int HM = W * RM, HN = 32 * RN, PLANE = HM * HN;
    constexpr int HALO = K;
    constexpr int TM = HM - 2 * HALO, TN = HN - 2 * HALO;
    static_assert(TM > 0 && TN > 0, "block depth too large for the tile");
    static_assert(sizeof(V) == 16 || K % 2 == 0, "complex64 tiles need an even halo (16-byte aligned TMA box origin)");
    static_assert(RN * sizeof(V) % 16 == 0, "a lane's row segment must be a whole number of 16-byte vectors");
    static_assert(K % RN == 0, "the halo must be a whole number of lane segments");
    static_assert(!(DIAG && OPEN), "the diagonal-lattice steps have no wall code (see step_diag)");

    extern __shared__ __align__(128) unsigned char smem_raw[];
    V *stage = reinterpret_cast<V *>(smem_raw);                    // stage[c][row][col]
    V *xch = stage + 4 * PLANE;                                    // xch[parity][warp][2 (diagonal: 4)][RN][32]
    uint64_t *bar = reinterpret_cast<uint64_t *>(xch + 2 * W * (DIAG ? 4 : 2) * RN * 32);   // "stage is full"
    uint64_t *xbar = bar + 2;                                      // xbar[parity][warp]: "slot of the warp is full"

    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const long long per_walk = (long long)a.tiles_m * a.tiles_n;
    constexpr int WORDS = sizeof(V) / 8;                           // the tensor map counts 8-byte words along n

    auto issue = [&](long long t) {                                // thread 0: TMA box loads of tile t, one per plane
        const long long w = t / per_walk;
        const long long r = t - w * per_walk;
        const int tm = a.tile_m0 + (int)(r / a.tiles_n), tn = a.tile_n0 + (int)(r % a.tiles_n);
        const int c0 = (tn * TN - HALO + a.ghost) * WORDS, c1 = tm * TM - HALO + a.ghost;
        t2d::mbar_expect_tx(bar, (uint32_t)(4 * PLANE * sizeof(V)));
#pragma unroll
        for (int c = 0; c < 4; ++c) t2d::tma_load_3d(stage + c * PLANE, &tmap, c0, c1, c * a.batch + (int)w, bar);
    };

    // does tile t write a site that can be non-zero?  (uniform over the CTA)
    auto active = [&](long long t) -> bool {
        if (a.dia_r < 0) return true;
        const long long r = t % per_walk;
        const long long lo_m = (long long)(a.tile_m0 + (int)(r / a.tiles_n)) * TM, lo_n = (long long)(a.tile_n0 + (int)(r % a.tiles_n)) * TN;
        const long long dm = a.dia_m < lo_m ? lo_m - a.dia_m : (a.dia_m > lo_m + TM - 1 ? a.dia_m - (lo_m + TM - 1) : 0);
        const long long dn = a.dia_n < lo_n ? lo_n - a.dia_n : (a.dia_n > lo_n + TN - 1 ? a.dia_n - (lo_n + TN - 1) : 0);
        return dm + dn <= a.dia_r;
    };
    auto next_active = [&](long long t) -> long long {
        while (t < a.total_tiles && !active(t)) t += gridDim.x;
        return t;
    };

    if (tid == 0) {
        t2d::mbar_init(bar, 1);
        for (int i = 0; i < 2 * W; ++i) t2d::mbar_init(xbar + i, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    long long t = next_active(blockIdx.x);
    if (tid == 0 && t < a.total_tiles) issue(t);
    const R *C = a.coin;                                           // kernel parameter = constant bank operands
    uint32_t phase = 0, xph = 0;

    for (long long t_next; t < a.total_tiles; t = t_next) {
        t_next = next_active(t + gridDim.x);
        const long long w = t / per_walk;
        const long long r = t - w * per_walk;
        const int tm = a.tile_m0 + (int)(r / a.tiles_n), tn = a.tile_n0 + (int)(r % a.tiles_n);
        const long long m0 = (long long)tm * TM - HALO, n0 = (long long)tn * TN - HALO;   // lattice coords of tile (0,0)
        const long long gm0 = m0 + wid * RM, gn0 = n0 + lane * RN;                        // ... of this lane's patch

        // ---- drain the stage into registers, then hand it to the prefetch of the next tile
        t2d::mbar_wait(bar, phase);
        phase ^= 1;
        t2d::Patch<R, RM, RN> p;
#pragma unroll
        for (int i = 0; i < RM; ++i) {
            const int off = (wid * RM + i) * HN + lane * RN;
            t2d::load_seg<RN>(stage + 0 * PLANE + off, p.c0[i]);
            t2d::load_seg<RN>(stage + 1 * PLANE + off, p.c1[i]);
            t2d::load_seg<RN>(stage + 2 * PLANE + off, p.c2[i]);
            t2d::load_seg<RN>(stage + 3 * PLANE + off, p.c3[i]);
        }
        __syncthreads();
        if (tid == 0 && t_next < a.total_tiles) issue(t_next);

        // ---- K steps in registers
        bool wall_tile = false;
        t2d::Walls wl = {-1, -1, -1, -1};
        if (OPEN) {
            wall_tile = (m0 <= 0) || (n0 <= 0) || (m0 + HM >= a.em) || (n0 + HN >= a.en);
            const long long il = -gm0, ir = a.em - 1 - gm0, jl = -gn0, jr = a.en - 1 - gn0;
            wl.il = (il >= 0 && il < RM) ? (int)il : -1;
            wl.ir = (ir >= 0 && ir < RM) ? (int)ir : -1;
            wl.jl = (jl >= 0 && jl < RN) ? (int)jl : -1;
            wl.jr = (jr >= 0 && jr < RN) ? (int)jr : -1;
        }
        if constexpr (DIAG)
            t2d::StepsDiag<R, RM, RN, W, KIND, 0, K>::run(p, C, a.coin_last, a.ratio, xch, xbar, xph, lane, wid);
        else
            t2d::Steps<R, RM, RN, W, KIND, OPEN, 0, K>::run(p, C, a.coin_last, a.ratio, xch, xbar, xph, lane, wid, wall_tile, wl);

        // ---- store the valid interior straight from registers: psi_c(i, j) after K steps sits at
        //      c0[i][(j-K) mod RN], c1[(i-K) mod RM][j], c2[(i+K) mod RM][j], c3[i][(j+K) mod RN]
        V *outw = a.out + w * a.walk_stride;
        const int lcol = lane * RN;
        const bool cols_in = (lcol >= HALO) && (lcol + RN <= HN - HALO);      // halo is a multiple of RN for RN = 2
#pragma unroll
        for (int i = 0; i < RM; ++i) {
            const int lrow = wid * RM + i;
            const long long gm = gm0 + i;
            if (lrow < HALO || lrow >= HM - HALO || gm >= a.em || !cols_in) continue;
            V *row = outw + gm * a.pitch + gn0;
            if (gn0 + RN <= a.en) {
                // whole segment inside the lattice: 16-byte vector stores
                cplx<R> z0[RN], z1[RN], z2[RN], z3[RN];
#pragma unroll
                for (int j = 0; j < RN; ++j) {
                    if constexpr (DIAG) {
                        z0[j] = p.c0[t2d_mod(i - K, RM)][t2d_mod(j - K, RN)];
                        z1[j] = p.c1[t2d_mod(i - K, RM)][t2d_mod(j + K, RN)];
                        z2[j] = p.c2[t2d_mod(i + K, RM)][t2d_mod(j - K, RN)];
                        z3[j] = p.c3[t2d_mod(i + K, RM)][t2d_mod(j + K, RN)];
                    } else {
                        z0[j] = p.c0[i][t2d_mod(j - K, RN)];
                        z1[j] = p.c1[t2d_mod(i - K, RM)][j];
                        z2[j] = p.c2[t2d_mod(i + K, RM)][j];
                        z3[j] = p.c3[i][t2d_mod(j + K, RN)];
                    }
                }
                t2d::store_seg<RN>(row + 0 * a.plane_stride, z0);
                t2d::store_seg<RN>(row + 1 * a.plane_stride, z1);
                t2d::store_seg<RN>(row + 2 * a.plane_stride, z2);
                t2d::store_seg<RN>(row + 3 * a.plane_stride, z3);
            } else {
#pragma unroll
                for (int j = 0; j < RN; ++j) {
                    if (gn0 + j < a.en) {
                        if constexpr (DIAG) {
                            cx_store<R>(row + 0 * a.plane_stride + j, p.c0[t2d_mod(i - K, RM)][t2d_mod(j - K, RN)]);
                            cx_store<R>(row + 1 * a.plane_stride + j, p.c1[t2d_mod(i - K, RM)][t2d_mod(j + K, RN)]);
                            cx_store<R>(row + 2 * a.plane_stride + j, p.c2[t2d_mod(i + K, RM)][t2d_mod(j - K, RN)]);
                            cx_store<R>(row + 3 * a.plane_stride + j, p.c3[t2d_mod(i + K, RM)][t2d_mod(j + K, RN)]);
                        } else {
                            cx_store<R>(row + 0 * a.plane_stride + j, p.c0[i][t2d_mod(j - K, RN)]);
                            cx_store<R>(row + 1 * a.plane_stride + j, p.c1[t2d_mod(i - K, RM)][j]);
                            cx_store<R>(row + 2 * a.plane_stride + j, p.c2[t2d_mod(i + K, RM)][j]);
                            cx_store<R>(row + 3 * a.plane_stride + j, p.c3[i][t2d_mod(j + K, RN)]);
                        }
                    }
                }
            }
        }
    }
}

}  // namespace qw
