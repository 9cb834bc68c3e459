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
};

template <typename R> __device__ __forceinline__ cplx<R> chain_shfl_down1(cplx<R> v) {
    v.re = __shfl_down_sync(0xffffffffu, v.re, 1);
    v.im = __shfl_down_sync(0xffffffffu, v.im, 1);
    return v;
}

// One walk step, U = step index inside the M-step period.  fw / fr: this tile's outflow record and the right
// neighbour's (entries 2U, 2U+1 of the current period).
template <typename R, int M, int KIND, int U>
__device__ __forceinline__ void chain1d_step(cplx<R> (&Rp)[M], cplx<R> (&Lp)[M], const R *C, int lane, bool has_in,
                                             typename Cx<R>::T *fw, const typename Cx<R>::T *fr) {
    typedef typename Cx<R>::T V;
#pragma unroll
    for (int q = 0; q < M; ++q) {
        const int p = (q + 2 * U) % M;
        cplx<R> v[2] = {Rp[q], Lp[p]};
        if constexpr (KIND == COIN_HADAMARD && M == 16) {
            // deferred scale, as in qw_step_blocked1d.cu: M-1 bare butterflies, then one scaled step with s^M
            if constexpr (U + 1 < M) {
                const cplx<R> r = v[0], l = v[1];
                v[0] = cx_add(r, l);
                v[1] = cx_sub(r, l);
            } else {
                apply_coin<R, 2, COIN_HADAMARD>(C + 1, v);      // C[1] = s^M
            }
        } else {
            apply_coin<R, 2, KIND>(C, v);
        }
        Rp[q] = v[0];
        Lp[p] = v[1];
    }
    // phi_L of logical sites 0 and 1 leaves the lane: it becomes L' of logical sites M-2, M-1 of the lane below
    // (lane 0: of the tile to the left, through the FIFO); lane 31 receives what the tile to the right recorded.
    constexpr int P0 = (2 * U) % M, P1 = (2 * U + 1) % M;
    const cplx<R> o0 = Lp[P0], o1 = Lp[P1];
    if (lane == 0) {
        V z0, z1;
        z0.x = o0.re; z0.y = o0.im; z1.x = o1.re; z1.y = o1.im;
        fw[2 * U] = z0; fw[2 * U + 1] = z1;
    }
    cplx<R> i0 = chain_shfl_down1(o0), i1 = chain_shfl_down1(o1);
    if (lane == 31 && has_in) {
        const V z0 = fr[2 * U], z1 = fr[2 * U + 1];
        i0 = cplx<R>{z0.x, z0.y}; i1 = cplx<R>{z1.x, z1.y};
    }
    Lp[P0] = i0;
    Lp[P1] = i1;
}

template <typename R, int M, int KIND, int U>
struct Chain1dUnroll {
    static __device__ __forceinline__ void run(cplx<R> (&Rp)[M], cplx<R> (&Lp)[M], const R *C, int lane, bool has_in,
                                               typename Cx<R>::T *fw, const typename Cx<R>::T *fr) {
        chain1d_step<R, M, KIND, U>(Rp, Lp, C, lane, has_in, fw, fr);
        if constexpr (U + 1 < M) Chain1dUnroll<R, M, KIND, U + 1>::run(Rp, Lp, C, lane, has_in, fw, fr);
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
    // warps per CTA x CTAs per SM: complex128 8 warps per SM, complex64 16
    static constexpr int WARPS = 4;
    static constexpr int MINB = sizeof(R) == 8 ? 2 : 4;
};

template <typename R, int M, int KIND>
__global__ void __launch_bounds__(Chain1dShape<R, M>::WARPS * 32, Chain1dShape<R, M>::MINB)
step_chain1d_kernel(const Chain1dArgs<R> a) {
    typedef typename Cx<R>::T V;
    constexpr int WARPS = Chain1dShape<R, M>::WARPS;
    constexpr int W = 32 * M;
    extern __shared__ __align__(16) unsigned char chain_smem[];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int per_warp = 3 * W + 4 * a.k;                                       // elements
    V *st_in = reinterpret_cast<V *>(chain_smem) + (size_t)wid * per_warp;      // [2][W]: prefetched input planes
    V *st_out = st_in + 2 * W;                                                  // [W]: output staging
    V *fifo = st_out + W;                                                       // [2][2k]: outflow records
    const long long N = a.n_sites;
    const long long G = (long long)gridDim.x * WARPS;

    R C[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) C[i] = a.coin[i];
    if constexpr (KIND == COIN_HADAMARD && M == 16) C[1] = a.scale_m;           // the (zero) imaginary part of C[0][0] is unused

    // element i*32 + lane of a tile: row (i*32 + lane) / M, col (i*32 + lane) % M
    int pos_co[M];                                                              // coalesced-side staging positions
#pragma unroll
    for (int i = 0; i < M; ++i) pos_co[i] = chain_pos<M, (int)sizeof(V)>((i * 32 + lane) / M, (i * 32 + lane) % M);

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
            for (int i = 0; i < M; ++i) chain_cp_async<(int)sizeof(V)>(st_in + pos_co[i], p0 + i * 32);
#pragma unroll
            for (int i = 0; i < M; ++i) chain_cp_async<(int)sizeof(V)>(st_in + W + pos_co[i], p1 + i * 32);
        } else {
#pragma unroll 1
            for (int plane = 0; plane < 2; ++plane) {
#pragma unroll 4
                for (int i = 0; i < M; ++i) {
                    long long x = X + i * 32 + lane;
                    if (x < 0) x += N; else if (x >= N) x -= N;
                    const int e = i * 32 + lane;                 // run-time i: not through the register array pos_co
                    chain_cp_async<(int)sizeof(V)>(st_in + plane * W + chain_pos<M, (int)sizeof(V)>(e / M, e % M),
                                                   inw + plane * a.plane_stride + x);
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
    while (chain < a.total_chains) {
        for (int j = 0; j <= nt; ++j) {
            const long long X = E - (long long)j * W;
            // ---- swizzled shared -> lane-contiguous registers
            cplx<R> Rp[M], Lp[M];
            asm volatile("cp.async.wait_group 0;" ::: "memory");
            __syncwarp();
#pragma unroll
            for (int i = 0; i < M; ++i) {
                const V zr = st_in[chain_pos<M, (int)sizeof(V)>(lane, i)], zl = st_in[W + chain_pos<M, (int)sizeof(V)>(lane, i)];
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
            // ---- k steps in registers; the outflow of this tile feeds the next one (its left neighbour)
            V *fw = fifo + (j & 1) * 2 * a.k;
            const V *fr = fifo + ((j & 1) ^ 1) * 2 * a.k;
            const bool has_in = j > 0;
            for (int s = 0; s < a.k; s += M) {
                Chain1dUnroll<R, M, KIND, 0>::run(Rp, Lp, C, lane, has_in, fw, fr);
                fw += 2 * M; fr += 2 * M;
            }
            __syncwarp();                                  // outflow record complete before the next tile reads it
            if (j == 0) continue;                          // the starter stores nothing
            // ---- store: element e of the tile is output site X + k + e; this chain owns input coordinates >= S
            const bool whole = X >= S && X + a.k + W <= N;
            const long long xo = X + a.k + lane;           // output coordinate of element `lane` (unwrapped)
#pragma unroll
            for (int plane = 0; plane < 2; ++plane) {
#pragma unroll
                for (int i = 0; i < M; ++i) {
                    V z;
                    if (plane == 0) { z.x = Rp[i].re; z.y = Rp[i].im; } else { z.x = Lp[i].re; z.y = Lp[i].im; }
                    st_out[chain_pos<M, (int)sizeof(V)>(lane, i)] = z;
                }
                __syncwarp();
                V *op = a.out + w * a.walk_stride + plane * a.plane_stride;
                if (whole) {
#pragma unroll
                    for (int i = 0; i < M; ++i) op[xo + i * 32] = st_out[pos_co[i]];
                } else {
#pragma unroll 4
                    for (int i = 0; i < M; ++i) {
                        long long x = xo + i * 32;
                        if (x - a.k >= S) {
                            if (x >= N) x -= N;
                            const int e = i * 32 + lane;
                            op[x] = st_out[chain_pos<M, (int)sizeof(V)>(e / M, e % M)];
                        }
                    }
                }
                __syncwarp();
            }
        }
        chain += G;
        if (chain < a.total_chains) chain_geom(chain, w, S, E, nt);
    }
}

// ---- host side ---------------------------------------------------------------------------------------------------

int chain1d_granule(const qw_sim *s) { return s->coin_kind == COIN_HADAMARD ? 16 : 8; }
constexpr int CHAIN1D_MAX_K = 64;       // FIFO size (4 k elements of shared memory per warp); also <= W/2 = 16*M
int chain1d_max_k(const qw_sim *) { return CHAIN1D_MAX_K; }

// Resident warps of the grid and the dynamic shared memory of one CTA at depth k.  The kernel attribute and the
// occupancy are taken once per device for the deepest launch, so every depth runs with the same persistent grid.
template <typename R, int M, int KIND>
static int chain1d_grid(const qw_sim *s, int k, int *warps_out, size_t *smem_out) {
    typedef typename Cx<R>::T V;
    constexpr int WARPS = Chain1dShape<R, M>::WARPS;
    const size_t smem_max = (size_t)WARPS * (3 * 32 * M + 4 * CHAIN1D_MAX_K) * sizeof(V);
    auto kern = step_chain1d_kernel<R, M, KIND>;
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
    *smem_out = (size_t)WARPS * (3 * 32 * M + 4 * k) * sizeof(V);
    return ctas_per_sm[dev];
}

template <typename R, int M, int KIND>
static int launch_chain1d_t(qw_sim *s, const void *in, void *out, int k, bool dry, double *cost) {
    typedef typename Cx<R>::T V;
    constexpr int WARPS = Chain1dShape<R, M>::WARPS;
    constexpr int W = 32 * M;
    const Geom &g = s->g;
    int grid_warps = 0; size_t smem = 0;
    if (chain1d_grid<R, M, KIND>(s, k, &grid_warps, &smem) < 1)
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
    for (int i = 0; i < M; ++i) sm = (R)(sm * a.coin[0]);    // s^M by repeated rounded products in the handle's precision
    a.scale_m = sm;
    long long blocks = (a.total_chains + WARPS - 1) / WARPS;
    if (blocks > grid_warps / WARPS) blocks = grid_warps / WARPS;
    step_chain1d_kernel<R, M, KIND><<<(unsigned)blocks, WARPS * 32, smem, s->stream>>>(a);
    QW_LAUNCH_CHECK(s, "step_chain1d_kernel");
    return QW_OK;
}

template <typename R>
static int launch_chain1d_r(qw_sim *s, const void *in, void *out, int k, bool dry, double *cost) {
    if (s->coin_kind == COIN_HADAMARD) return launch_chain1d_t<R, 16, COIN_HADAMARD>(s, in, out, k, dry, cost);
    return launch_chain1d_t<R, 8, COIN_GENERAL>(s, in, out, k, dry, cost);
}

// A ring with a uniform coin, at least two tiles long; k a multiple of the tile granule M, at most chain1d_max_k.
bool chain1d_eligible(const qw_sim *s, int k) {
    const Geom &g = s->g;
    const int M = chain1d_granule(s);
    return g.dim == 1 && g.boundary == QW_PERIODIC && s->coin_mode == QW_COIN_UNIFORM && !s->d_phases && !s->d_broken &&
           !s->rbl && g.en >= 64LL * M && k >= M && k % M == 0 && k <= chain1d_max_k(s);
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
