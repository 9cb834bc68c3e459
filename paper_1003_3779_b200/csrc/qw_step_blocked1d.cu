// qw_step_blocked1d.cu — temporally blocked 1D step: k applications of U = S (I (x) C)
// (eq. 2) per HBM round trip, for a uniform coin on a 1D lattice.
//
// Design: every WARP owns an independent tile of 32*M
// consecutive sites: valid = 32*M - 2k output sites plus a k-site halo on each side (after k steps
// the influence of the unknown outside has travelled exactly k sites inwards).
// Lane j keeps the M consecutive sites j*M .. j*M+M-1 of both coin planes in registers.  One step:
//   coin    in place on every (R[i], L[i]) pair                           (eq. 1)
//   shift   R moves one site right, L one site left (eq. 3).  Inside a lane this is a RENAMING
//           of registers, not a move: at step s logical site i lives in Rp[(i - s) mod M] and
//           Lp[(i + s) mod M]; only the element that crosses the lane boundary moves, through
//           one warp shuffle per plane.  The step loop is unrolled M times so every register
//           index is a compile-time constant; k must be a multiple of M.
// No block-level synchronisation and no shared-memory traffic inside the k steps; shared memory
// is only the staging area that turns coalesced global accesses into lane-contiguous registers.
// HBM bytes per site-step: coin_dim*sizeof(complex) * (32M/valid + 1) / k  instead of 2*coin_dim*sizeof(complex).
#include "qw_coin.cuh"

namespace qw {

constexpr int BLK1D_WARPS = 4;

template <typename R>
struct Blocked1dArgs {
    const typename Cx<R>::T *in;
    typename Cx<R>::T *out;
    long long n_sites;       // en
    long long walk_stride, plane_stride;
    long long tiles_per_walk, total_tiles;
    int k;                   // steps in this launch, multiple of M
    int valid;               // 32*M - 2k
    int boundary;
    R coin[8];
};

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

// One walk step with s = U (mod M).  x0 = unwrapped coordinate of this lane's logical site 0.
template <typename R, int M, int KIND, bool OPEN, int U>
__device__ __forceinline__ void blocked1d_step(cplx<R> (&Rp)[M], cplx<R> (&Lp)[M], const R *C,
                                               bool wall_warp, long long x0, long long n_sites) {
#pragma unroll
    for (int i = 0; i < M; ++i) {
        const int q = (i - U + M) % M, p = (i + U) % M;
        cplx<R> v[2] = {Rp[q], Lp[p]};
        apply_coin<R, 2, KIND>(C, v);
        Rp[q] = v[0];
        Lp[p] = v[1];
    }
    constexpr int QS = (M - 1 - U + M) % M;     // holds phi_R of logical M-1, becomes R' of logical 0
    constexpr int PS = U % M;                   // holds phi_L of logical 0,   becomes L' of logical M-1
    if constexpr (OPEN) {
        // reflecting walls (PAPER.md:94-101 with RBL = 0): R'[0] = phi_L[0], L'[N-1] = phi_R[N-1]
        if (wall_warp) {
            cplx<R> fixR = {0, 0}, fixL = {0, 0};
#pragma unroll
            for (int i = 0; i < M; ++i) {
                if (x0 + i == 0) fixR = Lp[(i + U) % M];
                if (x0 + i == n_sites - 1) fixL = Rp[(i - U + M) % M];
            }
            Rp[QS] = shfl_up1(Rp[QS]);
            Lp[PS] = shfl_down1(Lp[PS]);
#pragma unroll
            for (int i = 0; i < M; ++i) {
                if (x0 + i == 0) Rp[(i - U - 1 + 2 * M) % M] = fixR;
                if (x0 + i == n_sites - 1) Lp[(i + U + 1) % M] = fixL;
            }
            return;
        }
    }
    Rp[QS] = shfl_up1(Rp[QS]);
    Lp[PS] = shfl_down1(Lp[PS]);
}

template <typename R, int M, int KIND, bool OPEN, int U>
struct Blocked1dUnroll {
    static __device__ __forceinline__ void run(cplx<R> (&Rp)[M], cplx<R> (&Lp)[M], const R *C, bool wall_warp,
                                               long long x0, long long n_sites) {
        blocked1d_step<R, M, KIND, OPEN, U>(Rp, Lp, C, wall_warp, x0, n_sites);
        if constexpr (U + 1 < M) Blocked1dUnroll<R, M, KIND, OPEN, U + 1>::run(Rp, Lp, C, wall_warp, x0, n_sites);
    }
};

// padded staging position of tile element e (row = owning lane): odd row length -> conflict-free
template <int M> __device__ __forceinline__ int stage_pos(int e) { return (e / M) * (M + 1) + (e % M); }

template <typename R, int M, int KIND, bool OPEN>
__global__ void __launch_bounds__(BLK1D_WARPS * 32)
step_blocked1d_kernel(const Blocked1dArgs<R> a) {
    typedef typename Cx<R>::T V;
    __shared__ V stage[BLK1D_WARPS][32 * (M + 1)];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const long long tile_id = (long long)blockIdx.x * BLK1D_WARPS + wid;
    if (tile_id >= a.total_tiles) return;          // whole warp exits together
    const long long w = tile_id / a.tiles_per_walk;
    const long long t = tile_id - w * a.tiles_per_walk;
    const long long N = a.n_sites;
    const long long start = t * a.valid - a.k;     // unwrapped coordinate of tile element 0
    const V *inw = a.in + w * a.walk_stride;
    V *outw = a.out + w * a.walk_stride;
    V *st = stage[wid];

    cplx<R> Rp[M], Lp[M];
    // ---- load: coalesced global -> padded shared -> lane-contiguous registers, plane by plane
#pragma unroll
    for (int plane = 0; plane < 2; ++plane) {
        V tmp[M];
#pragma unroll
        for (int i = 0; i < M; ++i) {
            long long x = start + i * 32 + lane;
            bool ok = true;
            if (OPEN) ok = (x >= 0) && (x < N);
            else { if (x < 0) x += N; else if (x >= N) x -= N; }
            V z; z.x = 0; z.y = 0;
            if (ok) z = inw[plane * a.plane_stride + x];
            tmp[i] = z;
        }
#pragma unroll
        for (int i = 0; i < M; ++i) st[stage_pos<M>(i * 32 + lane)] = tmp[i];
        __syncwarp();
#pragma unroll
        for (int i = 0; i < M; ++i) {
            const V z = st[lane * (M + 1) + i];
            if (plane == 0) Rp[i] = cplx<R>{z.x, z.y}; else Lp[i] = cplx<R>{z.x, z.y};
        }
        __syncwarp();
    }

    // ---- k steps in registers
    R C[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) C[i] = a.coin[i];
    const long long x0 = start + (long long)lane * M;
    bool wall_warp = false;
    if (OPEN) wall_warp = (start <= 0) || (start + 32 * M >= N);
    for (int s = 0; s < a.k; s += M)
        Blocked1dUnroll<R, M, KIND, OPEN, 0>::run(Rp, Lp, C, wall_warp, x0, N);

    // ---- store the valid middle: registers -> padded shared -> coalesced global
#pragma unroll
    for (int plane = 0; plane < 2; ++plane) {
#pragma unroll
        for (int i = 0; i < M; ++i) {
            V z;
            if (plane == 0) { z.x = Rp[i].re; z.y = Rp[i].im; } else { z.x = Lp[i].re; z.y = Lp[i].im; }
            st[lane * (M + 1) + i] = z;
        }
        __syncwarp();
#pragma unroll
        for (int i = 0; i < M; ++i) {
            const int e = i * 32 + lane;
            const long long xo = t * a.valid + (e - a.k);       // unwrapped output site
            if (e >= a.k && e < 32 * M - a.k && xo < N)
                outw[plane * a.plane_stride + xo] = st[stage_pos<M>(e)];
        }
        __syncwarp();
    }
}

template <typename R, int M, int KIND>
static int launch_blocked1d_t(qw_sim *s, const void *in, void *out, int k) {
    typedef typename Cx<R>::T V;
    const Geom &g = s->g;
    Blocked1dArgs<R> a;
    a.in = static_cast<const V *>(in);
    a.out = static_cast<V *>(out);
    a.n_sites = g.en; a.walk_stride = g.walk_stride; a.plane_stride = g.plane_stride;
    a.k = k; a.valid = 32 * M - 2 * k;
    a.tiles_per_walk = (g.en + a.valid - 1) / a.valid;
    a.total_tiles = a.tiles_per_walk * g.batch;
    a.boundary = g.boundary;
    for (int i = 0; i < 8; ++i) a.coin[i] = (R)s->h_coin[i];
    const long long blocks = (a.total_tiles + BLK1D_WARPS - 1) / BLK1D_WARPS;
    if (blocks > 0x7fffffffLL) return fail(QW_EUNSUPPORTED, "lattice too large for one launch");
    if (g.boundary == QW_OPEN)
        step_blocked1d_kernel<R, M, KIND, true><<<(unsigned)blocks, BLK1D_WARPS * 32, 0, s->stream>>>(a);
    else
        step_blocked1d_kernel<R, M, KIND, false><<<(unsigned)blocks, BLK1D_WARPS * 32, 0, s->stream>>>(a);
    QW_LAUNCH_CHECK(s, "step_blocked1d_kernel");
    return QW_OK;
}

// Sites per lane: larger M = larger tiles (better valid fraction) but more registers and code.
template <typename R, int KIND> struct Blocked1dM { static constexpr int value = (KIND == COIN_HADAMARD) ? 16 : 8; };

int blocked1d_granule(const qw_sim *s) {
    return s->coin_kind == COIN_HADAMARD ? 16 : 8;
}

bool blocked1d_eligible(const qw_sim *s) {
    const Geom &g = s->g;
    return g.dim == 1 && s->coin_mode == QW_COIN_UNIFORM && !s->d_phases && !s->d_broken && !s->rbl &&
           g.en >= 32LL * blocked1d_granule(s);
}

int blocked1d_max_k(const qw_sim *s) {
    // keep at least half of every tile valid: 2k <= 16*M
    return 8 * blocked1d_granule(s);
}

int launch_step_blocked1d(qw_sim *s, const void *in, void *out, int k) {
    const int M = blocked1d_granule(s);
    if (k <= 0 || k % M != 0 || 2 * k >= 32 * M) return fail(QW_EINVAL, "blocked step depth %d invalid for tile granule %d", k, M);
    if (s->dtype == QW_C128) {
        if (s->coin_kind == COIN_HADAMARD) return launch_blocked1d_t<double, 16, COIN_HADAMARD>(s, in, out, k);
        return launch_blocked1d_t<double, 8, COIN_GENERAL>(s, in, out, k);
    }
    if (s->coin_kind == COIN_HADAMARD) return launch_blocked1d_t<float, 16, COIN_HADAMARD>(s, in, out, k);
    return launch_blocked1d_t<float, 8, COIN_GENERAL>(s, in, out, k);
}

}  // namespace qw
