// qw_step_chain1d.cu — temporally blocked 1D step on a RING without redundant halo work: k applications of
// U = S (I (x) C) (eq. 2) per HBM round trip, tiles chained through a stream of L amplitudes.
//
// Why a second blocked 1D kernel.  qw_step_blocked1d.cu gives every warp a tile with a k-site halo on each side that
// is recomputed by the neighbours: at k = 48 on 512-site tiles 19 % of the arithmetic is redundant.
// The two coin planes are pure advections (eq. 3: R moves +1, L moves -1 per step), so in the frame that
// MOVES WITH THE R PLANE nothing ever enters a tile from the left: a tile of W = 32*M sites that covers
// [X + t, X + t + W) at local step t keeps all its R amplitudes for all k steps; per step the two lowest L amplitudes
// leave through the left edge and two L amplitudes enter through the right edge — exactly the two that the tile to the
// right emitted at the same step.  A WARP therefore processes a CHAIN of adjacent tiles from right to left: while it
// advances tile j it records the 2k amplitudes that leave on the left in a FIFO (shared memory), and feeds them to
// tile j+1 (the left neighbour) one step at a time.  No tile computes a site twice.  Only the FIRST tile of a chain
// has no recorded stream: the warp first runs a "starter" tile immediately to the right of its chain whose own right
// inflow is garbage; the garbage front moves left 2 sites per step (relative to the tile), so for k <= W/2 the
// starter's left outflow is still exact.  Redundancy = one starter per chain = 1 / (tiles per chain), < 1 % on K1.
//
// Inside a tile (lane j keeps the M consecutive sites j*M .. j*M+M-1 of both planes in registers, as in the halo
// kernel): R never moves; the L plane moves 2 sites per step relative to the tile, which is a RENAMING of registers
// (logical site q of step t lives in Lp[(q + 2t) mod M]) plus two complex shuffles per step for the pair that
// crosses the lane boundary.  The M-step period is unrolled so that every register index is a compile-time constant.
// Tiles are staged through shared memory (coalesced cp.async in, coalesced stores out; XOR-swizzled, no padding),
// and the next tile of the chain is prefetched while the current one is advanced.
// After k steps the tile holds the sites [X + k, X + k + W): outputs are stored k sites to the right of the inputs.
//
// HBM bytes per site-step: coin_dim*sizeof(complex) * (2 + 1/tiles_per_chain) / k.
#include "qw_coin.cuh"
#include "qw_philox.cuh"

namespace qw {

template <typename R>
struct Chain1dArgs {
    const typename Cx<R>::T *in;
    typename Cx<R>::T *out;
    long long n_sites;       // ring length N
    long long walk_stride, plane_stride;
    long long chain_len;     // input sites per chain (a multiple of 32; the last chain of a walk may be shorter)
    long long total_chains;
    int chains_per_walk;
    int k;                   // steps in this launch: a multiple of M, <= 16*M
    R coin[8];
    R scale_m;               // deferred-scale Hadamard: s^M, applied once per M steps
    // random broken links redrawn every step (qw_set_random_broken_links; RBL template instances only)
    unsigned rbl_key0, rbl_key1;
    unsigned long long rbl_thr;     // floor(p * 2^32)
    unsigned t0;                    // step index of the first step of this launch (low 32 bits)
    // coin family (FAM template instances only; eq. 1): per-walk matrices and / or per-site phases
    const typename Cx<R>::T *coins;     // [walk][2][2], or nullptr (uniform coin)
    const typename Cx<R>::T *phases;    // [walk][site], or nullptr
};

// What the FAM instances carry through the steps: the phases of the lane's M sites (renamed like the L plane, one site
// per step: logical q of step t lives in ph[(q + t) mod M]) and where the next one comes from.
template <typename R, int M> struct Chain1dPhases {
    cplx<R> ph[M];
    const typename Cx<R>::T *row;   // phases of this walk
    long long next, n_sites;        // site whose phase enters the lane at the end of the current step
};

// What the RBL instances carry through the steps: the lattice coordinate of the lane's logical site 0 and the counter words.
struct Chain1dLinks {
    long long x0, n_sites;          // site of logical 0 of this lane at the current step (0 <= x0 < N); ring length
    unsigned t, walk, key0, key1;
    unsigned long long thr;
};

// ---- exchange by warp shuffles (complex64) -------------------------------------------------------------------------
template <typename R> __device__ __forceinline__ cplx<R> chain_shfl_from(cplx<R> v, int src) {
    v.re = __shfl_sync(0xffffffffu, v.re, src);
    v.im = __shfl_sync(0xffffffffu, v.im, src);
    return v;
}
// if (take) { a = p[0]; b = p[1]; } as predicated shared-memory loads INTO the registers that hold a and b
__device__ __forceinline__ void chain_fifo_load_in_place(const float2 *p, unsigned take, cplx<float> &a, cplx<float> &b) {
    const unsigned addr = (unsigned)__cvta_generic_to_shared(p);
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.u32 p, %4, 0;\n\t"
                 "@p ld.shared.v4.f32 {%0, %1, %2, %3}, [%5];\n\t}"
                 : "+f"(a.re), "+f"(a.im), "+f"(b.re), "+f"(b.im) : "r"(take), "r"(addr) : "memory");
}
__device__ __forceinline__ void chain_fifo_load_in_place(const double2 *p, unsigned take, cplx<double> &a, cplx<double> &b) {
    const unsigned addr = (unsigned)__cvta_generic_to_shared(p);
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.u32 p, %4, 0;\n\t"
                 "@p ld.shared.v2.f64 {%0, %1}, [%5];\n\t@p ld.shared.v2.f64 {%2, %3}, [%5+16];\n\t}"
                 : "+d"(a.re), "+d"(a.im), "+d"(b.re), "+d"(b.im) : "r"(take), "r"(addr) : "memory");
}

// ---- the exchange area -------------------------------------------------------------------------------------------
// Per step every lane hands the pair phi_L(logical site 0), phi_L(logical site 1) to the lane below.  This goes through
// shared memory, because there the FIFO costs nothing: addresses are per lane, so lane 0 simply writes its pair into the
// outflow record instead of the exchange row, and lane 31 reads the inflow record instead of the exchange row — no
// predicated instruction, no select, no register moves (warp shuffles cost 8 SHFL + about 12 MOV per step for
// complex128, measured: FP64 instructions occupy the issue port for two cycles each, so every other instruction is
// paid in FP64 time).  Addresses, in elements from the area base, for step t = s + U (U compile-time, s even):
//     exchange rows   B0 = [0, 32), B1 = B0 + P                      step parity U & 1 picks the row (WAR safety)
//     record a        [32, 32 + KMAX/2) for even t, + P for odd t     entry t at 32 + t/2 + (t & 1) * P
//     record b        [32 + KMAX/2, 32 + KMAX), + P for odd t          (tiles alternate between a and b)
// so every lane addresses  ptr + (U & 1) * P  with ptr a register that lane 0 / lane 31 bump by one element every
// second step and the other lanes never.  The first amplitude of a pair lives in area 0, the second in area 1.
// complex64 keeps the warp shuffles (4 SHFL per step and half as many FP instructions to hide them behind: measured
// faster, 5.4e12 against 4.8e12 site-updates/s on K1): there lane 0 saves its pair to the record [j & 1][2k], then loads
// the right-hand tile's pair into the same registers, and every lane takes the pair of lane + 1 (mod 32).
template <typename R> struct Chain1dExchange {
    static constexpr bool SMEM = sizeof(R) == 8;                  // exchange through shared memory (else shuffles)
    static constexpr int KMAX = sizeof(R) == 8 ? 96 : 128;      // deepest launch the records hold
    static constexpr int P = 32 + KMAX;                           // parity offset
    static constexpr int AREA = 2 * P;                            // elements per area; two areas
};

// One walk step, U = step index inside the M-step period.
//
// RBL (random broken links, eqs. 9-10): the link between the sites at logical positions Q and Q + 1
// carries phi_R[Q] to the right and phi_L[Q + 1] to the left; broken, both stay where they are with the opposite coin,
// i.e. the pair (R'[Q], L'[Q - 1]) = (phi_R[Q], phi_L[Q + 1]) is SWAPPED.  In this frame both members of the pair sit in
// the same lane — Rp[q] and the register that holds phi_L[q + 1] (for q = M - 1: the one just received from the lane
// above) — so a broken link is a predicated swap of two registers; its state is one Philox call per (site, step).
//
// FAM (coin family): phi = ph_x * (C_w psi) with the phase of the site (BASELINE.json:configs[4]).  The frame moves one
// site per step, so the lane's phases are renamed like a plane that moves one site per step, and the phase of the one site
// that enters the lane is read from global memory a step ahead (each phase is read once per tile: lane-strided, L2).
template <typename R, int M, int KIND, bool RBL, bool FAM, int U>
__device__ __forceinline__ void chain1d_step(cplx<R> (&Rp)[M], cplx<R> (&Lp)[M], const R *C,
                                             typename Cx<R>::T *&wptr, const typename Cx<R>::T *&rptr, int winc, int rinc,
                                             Chain1dLinks &lk, Chain1dPhases<R, FAM ? M : 1> &ps) {
    typedef typename Cx<R>::T V;
    typedef Chain1dExchange<R> EX;
    [[maybe_unused]] V ph_next;
    if constexpr (FAM) {
        if (ps.row) ph_next = ps.row[ps.next];
    }
#pragma unroll
    for (int q = 0; q < M; ++q) {
        const int p = (q + 2 * U) % M;
        cplx<R> v[2] = {Rp[q], Lp[p]};
        if constexpr (KIND == COIN_HADAMARD && M % 16 == 0) {
            // deferred scale, as in qw_step_blocked1d.cu: 15 bare butterflies, then one scaled step with s^16
            if constexpr (U % 16 != 15) {
                const cplx<R> r = v[0], l = v[1];
                v[0] = cx_add(r, l);
                v[1] = cx_sub(r, l);
            } else {
                apply_coin<R, 2, COIN_HADAMARD>(C + 1, v);      // C[1] = s^16
            }
        } else {
            apply_coin<R, 2, KIND>(C, v);
        }
        if constexpr (FAM) {
            if (ps.row) {
                const cplx<R> ph = ps.ph[(q + U) % (FAM ? M : 1)];
                v[0] = cx_mul(ph.re, ph.im, v[0]);
                v[1] = cx_mul(ph.re, ph.im, v[1]);
            }
        }
        Rp[q] = v[0];
        Lp[p] = v[1];
    }
    if constexpr (FAM) {
        if (ps.row) {                                             // logical site 0 leaves the lane, a new logical M-1 enters
            ps.ph[U % (FAM ? M : 1)] = cplx<R>{ph_next.x, ph_next.y};
            ps.next = ps.next + 1 == ps.n_sites ? 0 : ps.next + 1;
        }
    }
    constexpr int P0 = (2 * U) % M, P1 = (2 * U + 1) % M;
    // bit q of `bits`: the link owned by the site at logical position q (site x0 + q; in 1D link number = site index) is
    // broken at this step.  One generator call serves the four links 4g .. 4g+3 (reading R27), so a lane's M
    // consecutive sites need M/4 + 1 calls; a lane that straddles the seam of the ring takes one call per site.
    unsigned bits = 0;
    if constexpr (RBL) {
        if (lk.x0 + M <= lk.n_sites) {
            const unsigned long long g0 = (unsigned long long)lk.x0 >> 2;
            unsigned long long wide = 0;                           // bit 4 gi + wd: word wd of group g0 + gi
#pragma unroll
            for (int gi = 0; gi < M / 4 + 1; ++gi) {
                unsigned wd[4];
                rbl_group_words(g0 + gi, lk.t, lk.walk, lk.key0, lk.key1, wd);
#pragma unroll
                for (int i = 0; i < 4; ++i)
                    wide |= (unsigned long long)((unsigned long long)wd[i] < lk.thr ? 1u : 0u) << (4 * gi + i);
            }
            bits = (unsigned)(wide >> ((unsigned)lk.x0 & 3u));
        } else {
#pragma unroll 1
            for (int q = 0; q < M; ++q) {
                long long x = lk.x0 + q;
                if (x >= lk.n_sites) x -= lk.n_sites;
                bits |= ((unsigned long long)rbl_link_word((unsigned long long)x, lk.t, lk.walk, lk.key0, lk.key1) < lk.thr ? 1u : 0u) << q;
            }
        }
    }
    [[maybe_unused]] auto link_broken = [&](int q) -> bool { return (bits >> q) & 1u; };
    if constexpr (RBL) {
#pragma unroll
        for (int q = 0; q + 1 < M; ++q) {
            if (link_broken(q)) {
                const cplx<R> tmp = Rp[q];
                Rp[q] = Lp[(q + 1 + 2 * U) % M];
                Lp[(q + 1 + 2 * U) % M] = tmp;
            }
        }
    }
    // phi_L of logical sites 0 and 1 leaves the lane: it becomes L' of logical sites M-2, M-1 of the lane below
    V z0, z1;
    z0.x = Lp[P0].re; z0.y = Lp[P0].im; z1.x = Lp[P1].re; z1.y = Lp[P1].im;
    if constexpr (EX::SMEM) {
        constexpr int OFF = (U & 1) * EX::P;
        wptr[OFF] = z0;
        wptr[OFF + EX::AREA] = z1;
        __syncwarp();
        z0 = rptr[OFF];
        z1 = rptr[OFF + EX::AREA];
        Lp[P0] = cplx<R>{z0.x, z0.y};
        Lp[P1] = cplx<R>{z1.x, z1.y};
        if constexpr (U & 1) { wptr += winc; rptr += rinc; }      // lane 0 / lane 31: next pair of record entries
    } else {
        // winc != 0 marks lane 0; rinc = 1 if lane 0 takes a recorded inflow (not the starter), src lane in bits 8..
        cplx<R> o0 = Lp[P0], o1 = Lp[P1];
        if (winc) { wptr[2 * U] = z0; wptr[2 * U + 1] = z1; }
        chain_fifo_load_in_place(rptr + 2 * U, (unsigned)(rinc & 1), o0, o1);
        Lp[P0] = chain_shfl_from(o0, rinc >> 8);
        Lp[P1] = chain_shfl_from(o1, rinc >> 8);
    }
    if constexpr (RBL) {
        if (link_broken(M - 1)) {                                  // partner: what the lane above just handed over
            const cplx<R> tmp = Rp[M - 1];
            Rp[M - 1] = Lp[P0];
            Lp[P0] = tmp;
        }
        lk.t += 1;                                                 // next step: the frame has moved one site to the right
        lk.x0 = lk.x0 + 1 == lk.n_sites ? 0 : lk.x0 + 1;
    }
}

template <typename R, int M, int KIND, bool RBL, bool FAM, int U>
struct Chain1dUnroll {
    static __device__ __forceinline__ void run(cplx<R> (&Rp)[M], cplx<R> (&Lp)[M], const R *C,
                                               typename Cx<R>::T *&wptr, const typename Cx<R>::T *&rptr, int winc, int rinc,
                                               Chain1dLinks &lk, Chain1dPhases<R, FAM ? M : 1> &ps) {
        chain1d_step<R, M, KIND, RBL, FAM, U>(Rp, Lp, C, wptr, rptr, winc, rinc, lk, ps);
        if constexpr (U + 1 < M) Chain1dUnroll<R, M, KIND, RBL, FAM, U + 1>::run(Rp, Lp, C, wptr, rptr, winc, rinc, lk, ps);
    }
};

template <int BYTES>
__device__ __forceinline__ void chain_cp_async(void *smem_dst, const void *gmem_src) {
    const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    if constexpr (BYTES == 16)
        asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gmem_src) : "memory");
    else
        asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(d), "l"(gmem_src) : "memory");
}

// Staging position of tile element e = row * M + col (row = owning lane): XOR swizzle of the column with the row.
// Lane-contiguous accesses (lane = row, fixed col) and coalesced accesses (consecutive e) are both conflict-free for
// 16-byte (quarter warp per wavefront) and 8-byte (half warp) elements, without padding.  ES = element size.
// M = 8 with 8-byte elements: two rows share a 128-byte line, so the swizzle key is row / 2.
template <int M, int ES> __device__ __forceinline__ int chain_pos(int row, int col) {
    if constexpr (M == 8 && ES == 8) return row * M + (col ^ ((row >> 1) & 7));
    else return row * M + (col ^ (row & (M - 1)));
}

template <typename R, int M> struct Chain1dShape {
    // warps per CTA x CTAs per SM: complex128 8 warps per SM, complex64 12 (measured: 16 warps at 128 registers are slower)
#ifndef QW_CHAIN_M32
#define QW_CHAIN_M32 0      // 32 sites per lane for complex64 (8 warps per SM at 236 registers): measured 5.5e12 against 6.3e12 on K1
#endif
#ifndef QW_CHAIN_WARPS
#define QW_CHAIN_WARPS 4
#endif
#ifndef QW_CHAIN_MINB64
#define QW_CHAIN_MINB64 2
#endif
#ifndef QW_CHAIN_MINB32
#define QW_CHAIN_MINB32 3
#endif
    static constexpr int WARPS = QW_CHAIN_WARPS;
    static constexpr int MINB = (sizeof(R) == 8 || M == 32) ? QW_CHAIN_MINB64 : QW_CHAIN_MINB32;
    // shared memory of one warp, in elements: two prefetched input planes, HALF a plane of output staging, exchange
    static constexpr int SMEM_ELEMS = 2 * 32 * M + 16 * M +
        (Chain1dExchange<R>::SMEM ? 2 * Chain1dExchange<R>::AREA : 4 * Chain1dExchange<R>::KMAX);
};

template <typename R, int M, int KIND, bool RBL, bool FAM = false>
__global__ void __launch_bounds__(Chain1dShape<R, M>::WARPS * 32, Chain1dShape<R, M>::MINB)
step_chain1d_kernel(const Chain1dArgs<R> a) {
    typedef typename Cx<R>::T V;
    typedef Chain1dExchange<R> EX;
    constexpr int WARPS = Chain1dShape<R, M>::WARPS;
    constexpr int W = 32 * M;
    constexpr int ES = (int)sizeof(V);
    extern __shared__ __align__(16) unsigned char chain_smem[];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    V *st_in = reinterpret_cast<V *>(chain_smem) + (size_t)wid * Chain1dShape<R, M>::SMEM_ELEMS;   // [2][W]: prefetched input planes
    V *st_out = st_in + 2 * W;                                                  // [16][M]: output staging, half a plane
    V *area = st_out + 16 * M;                                                  // [2][AREA]: exchange rows + outflow records
    const long long N = a.n_sites;
    const long long G = (long long)gridDim.x * WARPS;

    R C[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) C[i] = a.coin[i];
    if constexpr (KIND == COIN_HADAMARD && M % 16 == 0) C[1] = a.scale_m;           // the (zero) imaginary part of C[0][0] is unused

    // element i*32 + lane of a tile: row (i*32 + lane) / M, col (i*32 + lane) % M
    int pos_co[M];                                                              // coalesced-side staging positions
#pragma unroll
    for (int i = 0; i < M; ++i) pos_co[i] = chain_pos<M, ES>((i * 32 + lane) / M, (i * 32 + lane) % M);

    // chain -> (walk, first input site S, end E, number of tiles); tile j of a chain starts at E - j*W (j = 0: starter)
    auto chain_geom = [&](long long c, long long &w, long long &S, long long &E, int &nt) {
        w = c / a.chains_per_walk;
        const long long ci = c - w * a.chains_per_walk;
        S = ci * a.chain_len;
        E = S + a.chain_len < N ? S + a.chain_len : N;
        nt = (int)((E - S + W - 1) / W);
    };
    // coalesced global -> swizzled shared, both planes of the tile that starts at unwrapped input coordinate X
    auto prefetch = [&](long long w, long long X) {
        const V *inw = a.in + w * a.walk_stride;
        if (X >= 0 && X + W <= N) {
            const V *p0 = inw + X + lane, *p1 = p0 + a.plane_stride;
#pragma unroll
            for (int i = 0; i < M; ++i) chain_cp_async<ES>(st_in + pos_co[i], p0 + i * 32);
#pragma unroll
            for (int i = 0; i < M; ++i) chain_cp_async<ES>(st_in + W + pos_co[i], p1 + i * 32);
        } else {
#pragma unroll 1
            for (int plane = 0; plane < 2; ++plane) {
#pragma unroll 4
                for (int i = 0; i < M; ++i) {
                    long long x = X + i * 32 + lane;
                    if (x < 0) x += N; else if (x >= N) x -= N;
                    const int e = i * 32 + lane;                 // run-time i: not through the register array pos_co
                    chain_cp_async<ES>(st_in + plane * W + chain_pos<M, ES>(e / M, e % M), inw + plane * a.plane_stride + x);
                }
            }
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
    };

    long long chain = (long long)blockIdx.x * WARPS + wid;
    long long w = 0, S = 0, E = 0;
    int nt = 0;
    if (chain < a.total_chains) {
        chain_geom(chain, w, S, E, nt);
        prefetch(w, E);
    }
    // exchange pointers of this lane (see Chain1dExchange): lanes 1..31 write row entry `lane`, lanes 0..30 read row
    // entry lane + 1; lane 0 writes and lane 31 reads the records, which alternate between a and b from tile to tile
    const int winc = lane == 0 ? 1 : 0, rinc = lane == 31 ? 1 : 0;
    while (chain < a.total_chains) {
        for (int j = 0; j <= nt; ++j) {
            const long long X = E - (long long)j * W;
            // ---- swizzled shared -> lane-contiguous registers
            cplx<R> Rp[M], Lp[M];
            asm volatile("cp.async.wait_group 0;" ::: "memory");
            __syncwarp();
#pragma unroll
            for (int i = 0; i < M; ++i) {
                const V zr = st_in[chain_pos<M, ES>(lane, i)], zl = st_in[W + chain_pos<M, ES>(lane, i)];
                Rp[i] = cplx<R>{zr.x, zr.y};
                Lp[i] = cplx<R>{zl.x, zl.y};
            }
            __syncwarp();
            // ---- prefetch the next tile of this chain, or the starter of this warp's next chain
            if (j < nt) {
                prefetch(w, X - W);
            } else if (chain + G < a.total_chains) {
                long long w2, S2, E2; int nt2;
                chain_geom(chain + G, w2, S2, E2, nt2);
                prefetch(w2, E2);
            }
            // ---- k steps in registers; the outflow of this tile is recorded for the next one (its left neighbour).
            // The starter (j = 0) reads a record nobody wrote: its inflow is garbage by construction.
            Chain1dPhases<R, FAM ? M : 1> ps;
            if constexpr (FAM) {
                if (a.coins) {                                     // the walk's own matrix (uniform otherwise)
                    const R *Cg = reinterpret_cast<const R *>(a.coins + w * 4);
#pragma unroll
                    for (int i = 0; i < 8; ++i) C[i] = Cg[i];
                }
                ps.row = a.phases ? a.phases + w * N : nullptr;
                ps.n_sites = N;
                long long x0 = X + (long long)lane * M;
                if (x0 < 0) x0 += N; else if (x0 >= N) x0 -= N;
                if (ps.row) {
#pragma unroll
                    for (int q = 0; q < M; ++q) {
                        long long x = x0 + q;
                        if (x >= N) x -= N;
                        const V z = ps.row[x];
                        ps.ph[q % (FAM ? M : 1)] = cplx<R>{z.x, z.y};
                    }
                }
                ps.next = x0 + M >= N ? x0 + M - N : x0 + M;
            }
            Chain1dLinks lk;
            if constexpr (RBL) {
                long long x0 = X + (long long)lane * M;            // X in (-W, N]: wrap once
                if (x0 < 0) x0 += N; else if (x0 >= N) x0 -= N;
                lk.x0 = x0; lk.n_sites = N; lk.t = a.t0; lk.walk = (unsigned)w;
                lk.key0 = a.rbl_key0; lk.key1 = a.rbl_key1; lk.thr = a.rbl_thr;
            }
            if constexpr (EX::SMEM) {
                V *wptr = area + (lane == 0 ? 32 + (j & 1) * (EX::KMAX / 2) : lane);
                const V *rptr = area + (lane == 31 ? 32 + ((j & 1) ^ 1) * (EX::KMAX / 2) : lane + 1);
                for (int s = 0; s < a.k; s += M)
                    Chain1dUnroll<R, M, KIND, RBL, FAM, 0>::run(Rp, Lp, C, wptr, rptr, winc, rinc, lk, ps);
            } else {
                V *wptr = area + (j & 1) * 2 * a.k;
                const V *rptr = area + ((j & 1) ^ 1) * 2 * a.k;
                const int rinc2 = (((lane + 1) & 31) << 8) | ((j > 0 && lane == 0) ? 1 : 0);
                for (int s = 0; s < a.k; s += M) {
                    Chain1dUnroll<R, M, KIND, RBL, FAM, 0>::run(Rp, Lp, C, wptr, rptr, winc, rinc2, lk, ps);
                    wptr += 2 * M; rptr += 2 * M;
                }
                __syncwarp();                              // outflow record complete before the next tile reads it
            }
            if (j == 0) continue;                          // the starter stores nothing
            // ---- store: element e of the tile is output site X + k + e; this chain owns input coordinates >= S.
            // Registers -> swizzled shared -> coalesced global, half a plane (the rows of 16 lanes) at a time.
            const bool whole = X >= S && X + a.k + W <= N;
#pragma unroll
            for (int plane = 0; plane < 2; ++plane) {
                V *op = a.out + w * a.walk_stride + plane * a.plane_stride;
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    __syncwarp();
                    if ((lane >> 4) == h) {
#pragma unroll
                        for (int i = 0; i < M; ++i) {
                            V z;
                            if (plane == 0) { z.x = Rp[i].re; z.y = Rp[i].im; } else { z.x = Lp[i].re; z.y = Lp[i].im; }
                            st_out[chain_pos<M, ES>(lane & 15, i)] = z;
                        }
                    }
                    __syncwarp();
                    const long long xo = X + a.k + h * (16 * M) + lane;      // output coordinate of half-plane element `lane`
                    if (whole) {
#pragma unroll
                        for (int i = 0; i < M / 2; ++i) op[xo + i * 32] = st_out[pos_co[i]];
                    } else {
#pragma unroll 4
                        for (int i = 0; i < M / 2; ++i) {
                            long long x = xo + i * 32;
                            if (x - a.k >= S) {
                                if (x >= N) x -= N;
                                const int e = i * 32 + lane;
                                op[x] = st_out[chain_pos<M, ES>(e / M, e % M)];
                            }
                        }
                    }
                }
            }
        }
        chain += G;
        if (chain < a.total_chains) chain_geom(chain, w, S, E, nt);
    }
}

// ---- host side ---------------------------------------------------------------------------------------------------

// a coin family the FAM instance handles: per-walk matrices and / or site phases on a general (not Hadamard-classified)
// matrix — the general evaluation, so that the result stays bit-identical to the generic kernel
static bool chain1d_family(const qw_sim *s) {
    if (s->coin_mode == QW_COIN_PER_WALK) return true;
    return s->coin_mode == QW_COIN_UNIFORM && s->d_phases != nullptr && s->coin_kind == COIN_GENERAL;
}
int chain1d_granule(const qw_sim *s) { return (s->coin_kind == COIN_HADAMARD && s->coin_mode == QW_COIN_UNIFORM) ? 16 : 8; }
// deepest launch: what the outflow records hold (Chain1dExchange::KMAX), and k <= W/2 = 16*M for the starter tile
int chain1d_max_k(const qw_sim *s) {
    const int kmax = s->dtype == QW_C128 ? Chain1dExchange<double>::KMAX : Chain1dExchange<float>::KMAX;
    const int half = 16 * chain1d_granule(s);
    return kmax < half ? kmax : half;
}

// Resident warps of the grid and the dynamic shared memory of one CTA at depth k.  The kernel attribute and the
// occupancy are taken once per device for the deepest launch, so every depth runs with the same persistent grid.
template <typename R, int M, int KIND, bool RBL, bool FAM>
static int chain1d_grid(const qw_sim *s, int k, int *warps_out, size_t *smem_out) {
    typedef typename Cx<R>::T V;
    constexpr int WARPS = Chain1dShape<R, M>::WARPS;
    const size_t smem_max = (size_t)WARPS * Chain1dShape<R, M>::SMEM_ELEMS * sizeof(V);
    auto kern = step_chain1d_kernel<R, M, KIND, RBL, FAM>;
    static int ctas_per_sm[64];                                            // per device (cudaFuncSetAttribute is per device)
    const int dev = s->device & 63;
    if (ctas_per_sm[dev] == 0) {
        if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_max) != cudaSuccess) {
            cudaGetLastError();
            return 0;
        }
        int n = 0;
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, kern, WARPS * 32, smem_max) != cudaSuccess) { cudaGetLastError(); return 0; }
        ctas_per_sm[dev] = n;
    }
    *warps_out = s->sm_count * ctas_per_sm[dev] * WARPS;
    *smem_out = smem_max;
    return ctas_per_sm[dev];
}

template <typename R, int M, int KIND, bool RBL, bool FAM = false>
static int launch_chain1d_t(qw_sim *s, const void *in, void *out, int k, bool dry, double *cost) {
    typedef typename Cx<R>::T V;
    constexpr int WARPS = Chain1dShape<R, M>::WARPS;
    constexpr int W = 32 * M;
    const Geom &g = s->g;
    int grid_warps = 0; size_t smem = 0;
    if (chain1d_grid<R, M, KIND, RBL, FAM>(s, k, &grid_warps, &smem) < 1)
        return fail(QW_ECUDA, "step_chain1d_kernel does not fit on an SM at depth %d", k);
    if (s->max_ctas > 0 && grid_warps > s->max_ctas * WARPS) grid_warps = s->max_ctas * WARPS;
    // chains: as many as the grid has warps (a multiple of them for a batch), each a multiple of 32 sites
    long long cpw = grid_warps / g.batch;
    if (cpw < 1) cpw = 1;
    long long len = (g.en + cpw - 1) / cpw;
    len = (len + 31) / 32 * 32;
    if (len < W) len = W;
    cpw = (g.en + len - 1) / len;
    if (cost) *cost = (double)((len + W - 1) / W + 1) * (double)((cpw * g.batch + grid_warps - 1) / grid_warps);
    if (dry) return QW_OK;
    Chain1dArgs<R> a;
    a.in = static_cast<const V *>(in);
    a.out = static_cast<V *>(out);
    a.n_sites = g.en; a.walk_stride = g.walk_stride; a.plane_stride = g.plane_stride;
    a.chain_len = len; a.chains_per_walk = (int)cpw; a.total_chains = cpw * g.batch;
    a.k = k;
    for (int i = 0; i < 8; ++i) a.coin[i] = (R)s->h_coin[i];
    R sm = (R)1;
    for (int i = 0; i < 16; ++i) sm = (R)(sm * a.coin[0]);   // s^16 by repeated rounded products in the handle's precision
    a.scale_m = sm;
    long long blocks = (a.total_chains + WARPS - 1) / WARPS;
    if (blocks > grid_warps / WARPS) blocks = grid_warps / WARPS;
    a.rbl_key0 = (unsigned)(s->rbl_seed & 0xffffffffu); a.rbl_key1 = (unsigned)(s->rbl_seed >> 32);
    a.rbl_thr = s->rbl_thr;
    a.t0 = (unsigned)((unsigned long long)s->t & 0xffffffffu);
    a.coins = s->coin_mode == QW_COIN_PER_WALK ? static_cast<const V *>(s->d_coin) : nullptr;
    a.phases = static_cast<const V *>(s->d_phases);
    step_chain1d_kernel<R, M, KIND, RBL, FAM><<<(unsigned)blocks, WARPS * 32, smem, s->stream>>>(a);
    QW_LAUNCH_CHECK(s, "step_chain1d_kernel");
    return QW_OK;
}

template <typename R>
static int launch_chain1d_r(qw_sim *s, const void *in, void *out, int k, bool dry, double *cost) {
    if (chain1d_family(s)) return launch_chain1d_t<R, 8, COIN_GENERAL, false, true>(s, in, out, k, dry, cost);
    if (s->rbl) {
        if (s->coin_kind == COIN_HADAMARD) return launch_chain1d_t<R, 16, COIN_HADAMARD, true>(s, in, out, k, dry, cost);
        return launch_chain1d_t<R, 8, COIN_GENERAL, true>(s, in, out, k, dry, cost);
    }
    if (s->coin_kind == COIN_HADAMARD) {
        // complex64: 32 sites per lane when the depth allows it (the register file holds twice as many complex64 sites;
        // half as many lane crossings and tile stagings per site)
        if constexpr (sizeof(R) == 4 && QW_CHAIN_M32) {
            if (k % 32 == 0 && s->g.en >= 64LL * 32) return launch_chain1d_t<R, 32, COIN_HADAMARD, false>(s, in, out, k, dry, cost);
        }
        return launch_chain1d_t<R, 16, COIN_HADAMARD, false>(s, in, out, k, dry, cost);
    }
    return launch_chain1d_t<R, 8, COIN_GENERAL, false>(s, in, out, k, dry, cost);
}

// A ring with a uniform coin, at least two tiles long; k a multiple of the tile granule M, at most chain1d_max_k.
bool chain1d_eligible(const qw_sim *s, int k) {
    const Geom &g = s->g;
    const int M = chain1d_granule(s);
    const bool plain = s->coin_mode == QW_COIN_UNIFORM && !s->d_phases;
    return g.dim == 1 && g.boundary == QW_PERIODIC && (plain || (chain1d_family(s) && !s->rbl)) && !s->d_broken &&
           g.en >= 64LL * M && k >= M && k % M == 0 && k <= chain1d_max_k(s);
}

// Tile computations per warp of one launch (the launch's cost in units of one tile advanced k steps).
double chain1d_cost(qw_sim *s, int k) {
    double c = 0.0;
    const int rc = s->dtype == QW_C128 ? launch_chain1d_r<double>(s, nullptr, nullptr, k, true, &c)
                                       : launch_chain1d_r<float>(s, nullptr, nullptr, k, true, &c);
    return rc == QW_OK ? c : 1e300;
}

int launch_step_chain1d(qw_sim *s, const void *in, void *out, int k) {
    return s->dtype == QW_C128 ? launch_chain1d_r<double>(s, in, out, k, false, nullptr)
                               : launch_chain1d_r<float>(s, in, out, k, false, nullptr);
}

}  // namespace qw
